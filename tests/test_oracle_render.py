"""Pins of the rendering oracle (oracle/render.py) against closed forms: a sphere's depth map and centre shade."""
import numpy as np

from oracle import render


def _sphere(n, R, width=1.0, hi=1.0, lo=0.1):
    z, y, x = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    c = (n - 1) / 2
    d = np.sqrt((x - c) ** 2 + (y - c) ** 2 + (z - c) ** 2)
    return 0.5 * (hi + lo) - 0.5 * (hi - lo) * np.tanh(2 * (d - R) / width), c


def test_sphere_depth_and_shade_closed_form():
    n, R = 48, 14.0
    rho, c = _sphere(n, R, width=4.0)          # a wide interface: linear interpolation between samples is accurate
    for axis in (0, 1, 2):
        shade, depth = render.render_isosurface(rho, 0.55, axis)
        v, u = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
        r2 = (u - c) ** 2 + (v - c) ** 2
        inside = r2 < (R - 3.0) ** 2
        exact = c - np.sqrt(np.maximum(R * R - r2, 0.0))            # first intersection of the ray with the sphere
        assert np.abs(depth[inside] - exact[inside]).max() < 0.05
        assert (depth[r2 > (R + 1.5) ** 2] == -1).all() and (shade[r2 > (R + 1.5) ** 2] == 0).all()
        # Lambert: shade = 0.1 + 0.9 max(0, n.l) with the sphere's outward normal
        nu, nv, nn = (u - c) / R, (v - c) / R, -np.sqrt(np.maximum(R * R - r2, 0.0)) / R
        lam = 0.1 + 0.9 * np.maximum(0.0, (nu + nv - 2 * nn) / np.sqrt(6))
        assert np.abs(shade[inside] - lam[inside]).max() < 0.02


def test_flat_layer_depth_is_exact_and_no_hit_is_empty():
    rho = np.full((16, 8, 8), 0.1)
    rho[10:, :, :] = 0.9                                             # jump between z = 9 and z = 10
    shade, depth = render.render_isosurface(rho, 0.5, 2, periodic=(True, True, False))
    assert np.allclose(depth, 9.5) and np.allclose(shade, 0.1 + 0.9 * 2 / np.sqrt(6))
    shade, depth = render.render_isosurface(np.full((8, 8, 8), 0.3), 0.5, 0)
    assert (depth == -1).all() and (shade == 0).all()


def test_tilted_plane_pins_axis_order_and_normal_sign():
    """dense phase behind the plane a.x = d, with three different slopes: the depth map and the shade are closed
    forms that change if two axes are exchanged or the normal's sign flips"""
    n = 40
    z, y, x = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    a = np.array([0.2, -0.35, 0.9]); a /= np.linalg.norm(a)          # unit normal (x, y, z) pointing into the dense phase
    s = a[0] * x + a[1] * y + a[2] * z - 14.0
    rho = 0.55 + 0.45 * np.tanh(s / 4.0)
    l = np.array([1.0, 1.0, -2.0]) / np.sqrt(6.0)
    for axis, (iu, iv) in ((2, (0, 1)), (1, (0, 2)), (0, (1, 2))):
        shade, depth = render.render_isosurface(rho, 0.55, axis, periodic=(False, False, False))
        v, u = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
        t = (14.0 - a[iu] * u - a[iv] * v) / a[axis]
        ok = (t > 2) & (t < n - 3) & (u > 0) & (u < n - 1) & (v > 0) & (v < n - 1)
        assert ok.sum() > 100
        assert np.abs(depth[ok] - t[ok]).max() < 0.02
        # the dense phase is where s > 0: its outward normal is -a; frame components (u, v, axis)
        nl = -(a[iu] * l[0] + a[iv] * l[1] + a[axis] * l[2])
        assert np.abs(shade[ok] - (0.1 + 0.9 * max(0.0, nl))).max() < 0.01
