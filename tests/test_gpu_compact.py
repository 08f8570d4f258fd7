"""GPU parity of the fluid-compact layout (lbm_compact.cuh): with at most a quarter of the cells fluid, lbm_step keeps
the populations in fluid-list order.  Against the oracle, against the dense list kernels (bit-identical), and across the
layout conversions that every export / import triggers."""
import os

import numpy as np
import pytest

from conftest import make_oracle
from paper_2506_17713_b200 import workloads as W
from test_gpu_parity import TOL16, TOL32, TOL64, assert_parity, fluid_mask, make_gpu, with_dtype

pytestmark = pytest.mark.gpu


def porous(dtype="f64", store=None, dims=(40, 28, 24)):
    """config 4's physics (two components, velocity inlet, pressure outlet) in a tighter seeded sphere pack"""
    wl, _ = W.config4(36, store_dtype="f32")
    nx, ny, nz = dims
    mask, _ = W.sphere_pack_mask(nx, ny, nz, porosity=0.12, rmin=3.0, rmax=7.0, buffer=3)
    assert 1.0 - mask.mean() <= 0.25
    wl = with_dtype(wl, dtype, store or dtype)
    wl.update(nx=nx, ny=ny, nz=nz)
    x = np.arange(nx * ny * nz) % nx
    nw = np.where(x < 3, 1.0, 0.03).astype(np.float32).astype(np.float64)
    w = np.where(x < 3, 0.03, 1.0).astype(np.float32).astype(np.float64)
    return wl, dict(rho=[nw, w], u=None, mask=mask)


def test_compact_fp64_against_the_oracle_with_exports_in_between():
    wl, inp = porous("f64")
    o, g = make_oracle(wl, inp), make_gpu(wl, inp)
    fl = fluid_mask(inp, o.N)
    for steps in (1, 40, 7, 33):
        o.step(steps); g.step(steps)
        assert g.hot_path == "two_pass_compact"
        fo = [o.get_populations(k) for k in range(2)]
        fg = [g.get_populations(k) for k in range(2)]          # compact -> dense -> compact round trip every time
        assert_parity(fo, fg, fl, TOL64, relative=False)
    ro, uo, po = o.get_macroscopic()
    rg, ug, pg = g.get_macroscopic()
    for k in range(2):
        assert np.abs(ro[k] - rg[k]).max() <= TOL64
        assert np.abs(o.get_psi(k) - g.get_psi(k)).max() <= TOL64
    assert np.abs(uo - ug).max() <= 1e-10 and np.abs(po - pg).max() <= TOL64
    # solid cells of the dense layout hold f_eq(1, 0) = w_i after a round trip (include/lbm.h, lbm_init_fields)
    from paper_2506_17713_b200 import binding
    e, w, opp = binding.get_lattice("D3Q19")
    assert np.abs(g.get_populations(0)[:, ~fl] - np.asarray(w)[:, None]).max() <= 1e-15


@pytest.mark.parametrize("dtype,store", [("f32", "f32"), ("f32", "f16"), ("f64", "f32")])
def test_compact_is_bit_identical_to_the_dense_list_kernels(dtype, store):
    wl, inp = porous(dtype, store)
    outs = []
    for compact in ("1", "0"):
        os.environ["LBM_TUNE_COMPACT"] = compact
        try:
            g = make_gpu(wl, inp)
            g.step(50)
            assert g.hot_path == ("two_pass_compact" if compact == "1" else "two_pass")
            outs.append([g.get_populations(k) for k in range(2)] + g.get_macroscopic()[0])
        finally:
            del os.environ["LBM_TUNE_COMPACT"]
    fl = fluid_mask(inp, outs[0][0].shape[-1])
    for a, b in zip(*outs):
        assert np.array_equal(a[..., fl], b[..., fl])


def test_compact_fp32_and_fp16_against_the_oracle():
    wl, inp = porous("f32", "f32")
    o, g = make_oracle(with_dtype(wl, "f64"), inp), make_gpu(wl, inp)
    o.step(100); g.step(100)
    assert g.hot_path == "two_pass_compact"
    assert_parity([o.get_populations(k) for k in range(2)], [g.get_populations(k) for k in range(2)], fluid_mask(inp, o.N), TOL32, relative=True)
    wl, inp = porous("f32", "f16")
    o, g = make_oracle(wl, inp), make_gpu(wl, inp)
    o.step(100); g.step(100)
    fl = fluid_mask(inp, o.N)
    for k in range(2):
        a, b = o.get_populations(k)[:, fl], g.get_populations(k)[:, fl]
        assert np.abs(a - b).max() <= TOL16 * np.abs(a).max()


def test_compact_d2q9_channels_and_pure_streaming():
    """D2Q9, two components, thin channels between thick walls (fluid fraction 3/16), walls on the y faces; with
    LBM_FLAG_NO_COLLIDE the step is a permutation and must be bit-exact"""
    wl, inp = W.config2(64, 32, "f64", wall=3)
    nx, ny = 64, 32
    mask = np.ones((ny, nx), np.uint8)
    mask[5:8, :] = 0
    mask[20:23, 4:60] = 0
    mask[8:20, 30:33] = 0                                          # a connecting throat
    inp = dict(inp, mask=mask.reshape(-1))
    assert 1.0 - mask.mean() <= 0.25
    o, g = make_oracle(wl, inp), make_gpu(wl, inp)
    o.step(60); g.step(60)
    assert g.hot_path == "two_pass_compact"
    fl = fluid_mask(inp, o.N)
    assert_parity([o.get_populations(k) for k in range(2)], [g.get_populations(k) for k in range(2)], fl, TOL64, relative=False)
    wl2 = dict(wl, no_collide=True)
    o, g = make_oracle(wl2, inp), make_gpu(wl2, inp)
    o.step(37); g.step(37)
    assert g.hot_path == "two_pass_compact"
    for k in range(2):
        assert np.array_equal(o.get_populations(k)[:, fl], g.get_populations(k)[:, fl])


def test_degenerate_masks_all_solid_and_single_fluid_cell():
    """nothing to update, and one fluid cell whose every link bounces back: mass stays put"""
    from paper_2506_17713_b200 import binding
    wl, inp = W.config5(16, "f64")
    e, w, opp = binding.get_lattice("D3Q19")
    N = 16 ** 3
    g = make_gpu(wl, dict(inp, mask=np.ones(N, np.uint8)))
    g.step(3)
    assert np.abs(g.get_populations(0) - np.asarray(w)[:, None]).max() <= 1e-15
    mask = np.ones(N, np.uint8)
    mask[5 + 16 * (6 + 16 * 7)] = 0
    inp1 = dict(inp, mask=mask)
    o, g = make_oracle(wl, inp1), make_gpu(wl, inp1)
    o.step(5); g.step(5)
    assert g.hot_path == "two_pass_compact"
    fl = mask == 0
    assert np.abs(o.get_populations(0)[:, fl] - g.get_populations(0)[:, fl]).max() <= TOL64
    assert abs(g.get_populations(0)[:, fl].sum() - np.asarray(inp["rho"][0])[fl].sum()) <= 1e-13
