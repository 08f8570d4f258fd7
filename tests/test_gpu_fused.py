"""GPU parity of the one-pass kernels K2F (k_fused_ws, k_fused_eq; D3Q19) against the oracle and against the two-pass path.

K2F recomputes rho -> psi of the ring around its tile instead of reading a psi field written by K1, so the
cases here stress what is new: tiles with ragged edges in x and y, several marching chunks, wrap-around of
the ring columns and rows, domains smaller than one tile, all dtype combinations it is built for, two
components, MRT and both forcing schemes.  Gates are those of test_gpu_parity.py.
"""
import numpy as np
import pytest

from conftest import make_oracle
from paper_2506_17713_b200 import workloads as W
from test_gpu_parity import TOL16, TOL32, TOL64, assert_parity, make_gpu, small_inputs, with_dtype

pytestmark = pytest.mark.gpu


def one_pass(wl):
    w = dict(wl)
    w["path"] = "one_pass"
    return w


def select_eq_kernel(monkeypatch, kernel):
    """k_fused_eq at full / half tile width, or k_fused_eq_split (built for fp32 compute and storage; other dtypes fall
    back to k_fused_eq) with the late / early take -- by the tuning knobs of include/lbm.h"""
    if kernel.startswith("k_fused_eq_split"):
        monkeypatch.setenv("LBM_TUNE_EQ_SPLIT", "2" if kernel.endswith("early") else "1")
    else:
        monkeypatch.setenv("LBM_TUNE_EQ_SPLIT", "0")
        monkeypatch.setenv("LBM_TUNE_EQ_HALF", "1" if kernel == "k_fused_eq_half" else "0")


def run_three(wl, inp, steps, oracle_wl=None):
    """oracle, K2F and the two-pass path on the same inputs; returns populations of each."""
    o = make_oracle(oracle_wl or wl, inp)
    g1 = make_gpu(one_pass(wl), inp)
    g2 = make_gpu(dict(wl, path="two_pass"), inp)
    o.step(steps)
    l0 = g1.kernel_launches
    g1.step(steps)
    assert g1.kernel_launches - l0 == steps      # one launch per step: K2F ran, not K1 + K2
    import os
    # k_fused_eq where the collision result is an equilibrium (one component, BGK, tau = 1), else k_fused_ws
    eq = wl["n_components"] == 1 and wl.get("collision", "BGK") == "BGK" and list(wl.get("tau", [1.0])) == [1.0] \
        and not os.environ.get("LBM_TUNE_NO_EQ")
    want = "one_pass_eq" if eq else "one_pass_ws"
    assert g1.hot_path == want, g1.hot_path        # and the intended kernel, not a silent fallback
    g2.step(steps)
    return ([o.get_populations(k) for k in range(o.nc)], [g1.get_populations(k) for k in range(o.nc)],
            [g2.get_populations(k) for k in range(o.nc)], o)


@pytest.mark.parametrize("kernel", ["k_fused_eq", "k_fused_eq_7_rows", "k_fused_eq_half", "k_fused_eq_split_late", "k_fused_eq_split_early",
                                    "k_fused_ws", "k_fused_ws_7_rows"])
@pytest.mark.parametrize("dims", [(128, 24, 20), (132, 9, 11), (4, 3, 2), (260, 8, 5), (8, 35, 3)])
def test_d3q19_fp64_ragged_tiles(dims, kernel, monkeypatch):
    monkeypatch.setenv("LBM_TUNE_FUSED_MCHUNK", "7")   # several marching chunks, ragged last one
    monkeypatch.setenv("LBM_TUNE_WS_TY", "7" if kernel.endswith("7_rows") else "8")   # rows per tile (plan_fused picks per domain)
    if kernel.startswith("k_fused_ws"):                 # the general kernel where k_fused_eq would apply
        monkeypatch.setenv("LBM_TUNE_NO_EQ", "1")
    else:
        select_eq_kernel(monkeypatch, "k_fused_eq" if kernel == "k_fused_eq_7_rows" else kernel)
    wl, _ = W.config5(16, "f64")
    wl.update(nx=dims[0], ny=dims[1], nz=dims[2])
    inp = small_inputs(wl, 21, 0.05, 0.3)
    fo, f1, f2, o = run_three(wl, inp, 30)
    fluid = np.ones(o.N, bool)
    assert_parity(fo, f1, fluid, TOL64, relative=False)
    assert_parity(f2, f1, fluid, 1e-13, relative=False)   # same arithmetic in the same order as K2


@pytest.mark.parametrize("kernel", ["k_fused_eq", "k_fused_eq_split_late", "k_fused_eq_split_early"])
@pytest.mark.parametrize("dims", [(128, 24, 20), (132, 9, 11), (4, 3, 2), (260, 8, 5), (8, 35, 3), (200, 17, 9)])
def test_d3q19_fp32_ragged_tiles(dims, kernel, monkeypatch):
    """fp32 compute and storage (what k_fused_eq_split is built for): ragged tiles in x and y, chunks with a ragged tail,
    domains smaller than a tile or a half row; against the fp64 oracle and the two-pass path."""
    monkeypatch.setenv("LBM_TUNE_FUSED_MCHUNK", "7")
    select_eq_kernel(monkeypatch, kernel)
    wl, _ = W.config5(16, "f32")
    wl.update(nx=dims[0], ny=dims[1], nz=dims[2])
    inp = small_inputs(wl, 22, 0.05, 0.3)
    fo, f1, f2, o = run_three(wl, inp, 30, oracle_wl=with_dtype(wl, "f64"))
    fluid = np.ones(o.N, bool)
    assert_parity(fo, f1, fluid, TOL32, relative=True)
    assert_parity(f2, f1, fluid, 2e-6, relative=True)    # same arithmetic as K1 / K2 (fp32: up to contraction of a*b+c)


@pytest.mark.parametrize("kernel", ["k_fused_eq", "k_fused_eq_half", "k_fused_eq_split_late", "k_fused_eq_split_early", "k_fused_ws",
                                    "k_fused_ws_7_rows"])
def test_config5_fp32_100_steps(kernel, monkeypatch):
    if kernel.startswith("k_fused_ws"):
        monkeypatch.setenv("LBM_TUNE_NO_EQ", "1")
        monkeypatch.setenv("LBM_TUNE_WS_TY", "7" if kernel.endswith("7_rows") else "8")
    else:
        select_eq_kernel(monkeypatch, kernel)
    wl, inp = W.config5(48, "f32")
    fo, f1, f2, o = run_three(wl, inp, 100, oracle_wl=with_dtype(wl, "f64"))
    fluid = np.ones(o.N, bool)
    assert_parity(fo, f1, fluid, TOL32, relative=True)
    assert_parity(f2, f1, fluid, 2e-6, relative=True)


@pytest.mark.parametrize("dims,dtype,store", [((136, 26, 12), "f64", "f64"), ((264, 27, 10), "f32", "f32"),
                                              ((272, 26, 9), "f32", "f16"), ((136, 34, 7), "f64", "f32")])
def test_d3q19_several_tiles_all_dtypes(dims, dtype, store, monkeypatch):
    """Domains several tiles wide and tall (tiles on and off the periodic seams, ragged last tiles), every dtype
    combination the warp-specialised kernel is built for."""
    monkeypatch.setenv("LBM_TUNE_FUSED_MCHUNK", "5")
    wl, _ = W.config5(16, dtype, store_dtype=store)
    wl.update(nx=dims[0], ny=dims[1], nz=dims[2])
    inp = small_inputs(wl, 31, 0.05, 0.3)
    steps = 30
    fo, f1, f2, o = run_three(wl, inp, steps, oracle_wl=None if dtype == "f64" and store == "f64" else with_dtype(wl, "f64") if store != "f16" else None)
    fluid = np.ones(o.N, bool)
    if store == "f16":
        assert_parity(fo, f1, fluid, TOL16, relative=True)      # oracle emulates the fp16 rounding at the store
    elif dtype == "f64" and store == "f64":
        assert_parity(fo, f1, fluid, TOL64, relative=False)
        assert_parity(f2, f1, fluid, 1e-13, relative=False)
    elif dtype == "f64":                                          # fp64 compute, fp32 storage
        assert_parity(f2, f1, fluid, 1e-6, relative=True)
    else:
        assert_parity(fo, f1, fluid, TOL32, relative=True)


def test_two_components_several_tiles_fp32():
    g = 3.5 / 3.0
    wl = dict(name="x", lattice="D3Q19", nx=140, ny=26, nz=7, n_components=2, periodic=(True, True, True),
              psi_kind=["SC93", "SC93"], eos=[dict(rho0=1.0), dict(rho0=1.0)], G=[[0.0, g], [g, 0.0]],
              collision="BGK", tau=[1.0, 1.0], forcing="EDM", compute_dtype="f32", store_dtype="f32")
    inp = small_inputs(wl, 6, 0.4, 0.9)
    fo, f1, f2, o = run_three(wl, inp, 30, oracle_wl=with_dtype(wl, "f64"))
    assert_parity(fo, f1, np.ones(o.N, bool), TOL32, relative=True)


def test_config5_fp16_storage():
    wl, inp = W.config5(32, "f32", store_dtype="f16")
    fo, f1, f2, o = run_three(wl, inp, 100)   # the oracle emulates the fp16 rounding at the store (R16)
    fluid = np.ones(o.N, bool)
    assert_parity(fo, f1, fluid, TOL16, relative=True)


@pytest.mark.parametrize("rows", [8, 7])
def test_config3_mrt_peng_robinson_fp64(rows, monkeypatch):
    monkeypatch.setenv("LBM_TUNE_WS_TY", str(rows))     # rows per tile of k_fused_ws (7 on 256^3: every SM gets a CTA)
    wl, _ = W.config3(20, "f64")
    wl.update(nx=24, ny=19, nz=17)
    inp = small_inputs(wl, 3, 3.9, 4.2)
    fo, f1, f2, o = run_three(wl, inp, 100)
    assert_parity(fo, f1, np.ones(o.N, bool), TOL64, relative=False)


@pytest.mark.parametrize("lattice,n", [("D3Q19", (24, 10, 9)), ("D3Q19", (136, 19, 6))])
@pytest.mark.parametrize("collision", ["BGK", "MRT"])
@pytest.mark.parametrize("forcing", ["EDM", "SHIFT"])
def test_two_components_variants_fp32(lattice, n, collision, forcing):
    g = 3.5 / 3.0
    wl = dict(name="x", lattice=lattice, nx=n[0], ny=n[1], nz=n[2], n_components=2, periodic=(True, True, True),
              psi_kind=["SC93", "RHO"], eos=[dict(rho0=1.0), dict()], G=[[-0.3, g * 0.4], [g * 0.4, 0.0]],
              collision=collision, tau=[0.8, 1.3], forcing=forcing, compute_dtype="f32", store_dtype="f32")
    if collision == "MRT":
        wl["mrt_rates"] = [W.mrt_rates(lattice, 0.8), W.mrt_rates(lattice, 1.3)]
    inp = small_inputs(wl, 5, 0.4, 0.9)
    fo, f1, f2, o = run_three(wl, inp, 100, oracle_wl=with_dtype(wl, "f64"))
    assert_parity(fo, f1, np.ones(o.N, bool), TOL32, relative=True)


def test_one_pass_refused_where_it_does_not_apply():
    from paper_2506_17713_b200 import binding
    wl, inp = W.config2(64, 32, "f32", wall=3)          # solid plates
    s = make_gpu(one_pass(wl), inp)
    with pytest.raises(binding.LBMError):
        s.step(1)
    wl, inp = W.config5(16, "f32")
    wl.update(nx=18)                                     # rows that are not whole 16-byte vectors
    inp = small_inputs(wl, 1)
    s = make_gpu(one_pass(wl), inp)
    with pytest.raises(binding.LBMError):
        s.step(1)
    wl, inp = W.config1(32, "f64")                       # D2Q9: no one-pass kernel (the two-pass path wins there)
    s = make_gpu(one_pass(wl), inp)
    with pytest.raises(binding.LBMError):
        s.step(1)


@pytest.mark.parametrize("dims,ygroup,mchunk,take", [((128, 40, 30), 2, 8, "late"), ((200, 17, 9), 1, 4, "early"), ((132, 70, 21), 3, 21, "late")])
def test_split_kernel_launched_per_chunk_and_row_group(dims, ygroup, mchunk, take, monkeypatch):
    """k_fused_eq_split launched once per chunk of planes and per group of tile rows (what lbm_step does on domains whose tile
    columns are one wave, e.g. 384^3: lbm_api.cu plan_fused): ragged last group and last chunk; bit-identical to the single
    launch, every launch counted, and within the fp32 gate of the oracle."""
    from paper_2506_17713_b200 import binding
    wl, _ = W.config5(16, "f32")
    wl.update(nx=dims[0], ny=dims[1], nz=dims[2])
    inp = small_inputs(wl, 31, 0.05, 0.3)
    monkeypatch.setenv("LBM_TUNE_FUSED_MCHUNK", str(mchunk))
    monkeypatch.setenv("LBM_TUNE_EQ_SPLIT", "2" if take == "early" else "1")
    out = {}
    for grouped in (True, False):
        if grouped:
            monkeypatch.setenv("LBM_TUNE_EQ_YGROUP", str(ygroup))
        else:
            monkeypatch.delenv("LBM_TUNE_EQ_YGROUP", raising=False)
        g = make_gpu(one_pass(wl), inp)
        l0 = g.kernel_launches
        g.step(20)
        assert g.hot_path == "one_pass_eq"
        per_step = 1
        if grouped:
            yt = (dims[1] + 7) // 8
            per_step = ((dims[2] + mchunk - 1) // mchunk) * ((yt + ygroup - 1) // ygroup)
        assert g.kernel_launches - l0 == 20 * per_step
        out[grouped] = g.get_populations(0)
    assert np.array_equal(out[True], out[False])
    o = make_oracle(with_dtype(wl, "f64"), inp)
    o.step(20)
    assert_parity([o.get_populations(0)], [out[True]], np.ones(o.N, bool), TOL32, relative=True)


@pytest.mark.parametrize("dims,collision", [((128, 1120, 40), "BGK"),    # 140 tile columns: one wave, one chunk
                                            ((256, 560, 200), "BGK"),    # 140 columns, two launches of 100 planes
                                            ((256, 256, 40), "MRT"),     # k_fused_ws, 7- against 8-row tiles by the planner
                                            ((416, 104, 60), "BGK"),     # ragged last x tile: planes per CTA from the play-through
                                            ((384, 296, 24), "MRT")])
def test_default_launch_plans_match_the_two_pass_path(dims, collision):
    """Whatever plan_fused picks for a domain (tile height, planes per CTA, a launch per chunk): the one-pass result equals
    the two-pass path's to fp32 contraction, on domains large enough to reach those rules (no tuning knob set)."""
    wl, _ = W.config5(16, "f32")
    wl.update(nx=dims[0], ny=dims[1], nz=dims[2], collision=collision)
    if collision == "MRT":
        wl["mrt_rates"] = [W.mrt_rates("D3Q19", 1.0)]
    inp = small_inputs(wl, 41, 0.05, 0.3)
    g1 = make_gpu(wl, inp)
    g2 = make_gpu(dict(wl, path="two_pass"), inp)
    g1.step(5)
    g2.step(5)
    assert g1.hot_path in ("one_pass_eq", "one_pass_ws"), g1.hot_path
    assert g2.hot_path == "two_pass"
    f1, f2 = g1.get_populations(0), g2.get_populations(0)
    assert np.isfinite(f1).all()
    assert np.abs(f1 - f2).max() <= 2e-6 * np.abs(f2).max()
