"""ORACLE -- TEST INFRASTRUCTURE ONLY.  CPU restatement of the headless iso-surface rendering of a density field
(the paper renders GPU-resident arrays in situ with a third-party tool, and
gives no formula, so this file IS the definition).  Plain numpy, fp64, shares no code with
the CUDA path.

Orthographic rays along +axis through rho[z, y, x].  Pixel (u, v) = the two other axes in ascending order.  Along a
ray the first sample pair (k, k+1) with (rho_k - iso)(rho_{k+1} - iso) <= 0 and rho_k != rho_{k+1} is the hit:
depth t = k + (iso - rho_k) / (rho_{k+1} - rho_k); no hit: depth = -1, shade = 0.  Shade = 0.1 + 0.9 max(0, n.l) with
n = -grad(rho) / |grad(rho)| (outward normal of the dense phase; central differences with periodic wrap or clamped
indices, interpolated linearly between the two samples) and the light direction l = (1, 1, -2) / sqrt(6) in the
(u, v, axis) frame (towards the viewer, who looks along +axis); |grad| = 0 gives shade 0.1.
"""
import numpy as np


def _grad(rho, periodic):
    """central differences, components ordered (x, y, z); clamped indices on non-periodic axes"""
    g = []
    for ax_np, per in ((2, periodic[0]), (1, periodic[1]), (0, periodic[2])):
        n = rho.shape[ax_np]
        idx = np.arange(n)
        ip = (idx + 1) % n if per else np.minimum(idx + 1, n - 1)
        im = (idx - 1) % n if per else np.maximum(idx - 1, 0)
        g.append(0.5 * (np.take(rho, ip, axis=ax_np) - np.take(rho, im, axis=ax_np)))
    return g   # gx, gy, gz


def render_isosurface(rho, iso, axis, periodic=(True, True, True)):
    """rho: array [nz, ny, nx]; returns (shade [n_v, n_u], depth [n_v, n_u])"""
    rho = np.asarray(rho, dtype=np.float64)
    gx, gy, gz = _grad(rho, periodic)
    # bring the marching axis first: arrays [n_a, n_v, n_u]; frame components (u, v, a)
    if axis == 2:
        r, gu, gv, ga = rho, gx, gy, gz                              # u = x, v = y
    elif axis == 1:
        tr = lambda a: np.transpose(a, (1, 0, 2))                     # [y, z, x]: u = x, v = z
        r, gu, gv, ga = tr(rho), tr(gx), tr(gz), tr(gy)
    else:
        tr = lambda a: np.transpose(a, (2, 0, 1))                     # [x, z, y]: u = y, v = z
        r, gu, gv, ga = tr(rho), tr(gy), tr(gz), tr(gx)
    na = r.shape[0]
    shade = np.zeros(r.shape[1:])
    depth = np.full(r.shape[1:], -1.0)
    done = np.zeros(r.shape[1:], dtype=bool)
    l = np.array([1.0, 1.0, -2.0]) / np.sqrt(6.0)
    for k in range(na - 1):
        a, b = r[k], r[k + 1]
        hit = (~done) & ((a - iso) * (b - iso) <= 0) & (a != b)
        if not hit.any():
            continue
        w = np.where(hit, (iso - a) / np.where(a != b, b - a, 1.0), 0.0)
        nu = -((1 - w) * gu[k] + w * gu[k + 1])
        nv = -((1 - w) * gv[k] + w * gv[k + 1])
        nn = -((1 - w) * ga[k] + w * ga[k + 1])
        norm = np.sqrt(nu * nu + nv * nv + nn * nn)
        dot = np.where(norm > 0, (nu * l[0] + nv * l[1] + nn * l[2]) / np.where(norm > 0, norm, 1.0), 0.0)
        shade = np.where(hit, 0.1 + 0.9 * np.maximum(0.0, dot), shade)
        depth = np.where(hit, k + w, depth)
        done |= hit
    return shade, depth
