"""GPU parity of lbm_render_isosurface (in-situ rendering) against oracle/render.py: the CUDA kernel
renders the resident density field; the oracle renders the field the same handle exports."""
import numpy as np
import pytest

from oracle import render
from paper_2506_17713_b200 import workloads as W
from conftest import make_oracle
from test_gpu_parity import make_gpu, small_inputs

pytestmark = pytest.mark.gpu


def _field(g, k=0):
    c = g.cfg
    return g.get_macroscopic(want_u=False, want_p=False)[0][k].reshape(c.nz, c.ny, c.nx)


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_droplets_fp64_every_axis(axis):
    wl, inp = W.config5(32, "f64")
    o, g = make_oracle(wl, inp), make_gpu(wl, inp)
    o.step(20); g.step(20)
    iso = 0.5 * (W.CS_RHO_L_085 + W.CS_RHO_V_085)
    shade, depth = g.render_isosurface(iso, axis)
    so, do = render.render_isosurface(_field(g), iso, axis)
    assert (depth >= 0).sum() > 20 and (depth < 0).sum() > 20           # droplets and empty background both in view
    assert np.array_equal(depth < 0, do < 0)
    assert np.abs(depth - do).max() <= 1e-11 and np.abs(shade - so).max() <= 1e-10
    # and against the field of the oracle's own state
    so2, do2 = render.render_isosurface(o.get_macroscopic()[0][0].reshape(32, 32, 32), iso, axis)
    assert np.array_equal(depth < 0, do2 < 0) and np.abs(depth - do2).max() <= 1e-8 and np.abs(shade - so2).max() <= 1e-7
    g.step(3)                                                           # the scratch images did not disturb the state
    o.step(3)
    assert np.abs(g.get_populations(0) - o.get_populations(0)).max() <= 1e-12


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_non_cubic_box_pins_the_pixel_order(dtype):
    wl, _ = W.config5(16, dtype)
    wl.update(nx=40, ny=12, nz=9)
    inp = small_inputs(wl, 23, 0.05, 0.3)
    g = make_gpu(wl, inp)
    g.step(5)
    for axis, shape in ((2, (12, 40)), (1, (9, 40)), (0, (9, 12))):
        shade, depth = g.render_isosurface(0.1875, axis)                # representable in fp32
        assert shade.shape == shape
        so, do = render.render_isosurface(_field(g), 0.1875, axis)
        assert np.array_equal(depth < 0, do < 0)
        tol = 1e-11 if dtype == "f64" else 2e-4
        assert np.abs(depth - do).max() <= tol and np.abs(shade - so).max() <= 10 * tol


def test_two_components_with_walls_2d_and_clamped_axes():
    wl, inp = W.config2(64, 32, "f64", wall=3)
    g = make_gpu(wl, inp)
    g.step(10)
    per = tuple(bool(p) for p in wl["periodic"]) + (True,) * (3 - len(wl["periodic"]))
    for k in (0, 1):
        f = _field(g, k)
        iso = 0.5 * (f.max() + f[f > 0].min())
        for axis in (0, 1):
            shade, depth = g.render_isosurface(iso, axis, k=k, dtype=np.float32)
            so, do = render.render_isosurface(f, iso, axis, periodic=per)
            assert (do >= 0).any()
            assert np.array_equal(depth < 0, do < 0)
            assert np.abs(depth - do).max() <= 1e-5 and np.abs(shade - so).max() <= 1e-5   # fp32 images of fp64 arithmetic


def test_render_argument_errors():
    from paper_2506_17713_b200 import binding
    wl, inp = W.config1(64, "f64")
    g = binding.LBM(wl)
    with pytest.raises(binding.LBMError):
        g.render_isosurface(0.5, 0)                                     # before init_fields
    g = make_gpu(wl, inp)
    with pytest.raises(binding.LBMError):
        g.render_isosurface(0.5, 3)
    with pytest.raises(binding.LBMError):
        g.render_isosurface(0.5, 0, k=1)
