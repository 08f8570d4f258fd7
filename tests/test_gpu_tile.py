"""k_steps_tile (lbm_small.cuh): the tiled persistent kernel of small 2-D domains against the plain launches of the two-pass
kernels, bit for bit, on the shapes that stress its ring logic -- domains narrower than a ring, ragged tiles, walls inside
the ring, non-periodic faces with velocity / pressure rules, several tile sizes, every dtype pair and collision -- and
against the oracle within the tolerances of test_gpu_parity.py.
"""
import numpy as np
import pytest

from conftest import make_oracle
from paper_2506_17713_b200 import workloads as W
from test_gpu_parity import TOL32, TOL64, assert_parity, fluid_mask, small_inputs, with_dtype

pytestmark = pytest.mark.gpu


def run_gpu(wl, inp, calls, monkeypatch, plain):
    """The populations after the given lbm_step calls: on the default path (k_steps_tile), or step by step (plain launches)."""
    from paper_2506_17713_b200 import binding
    for v in ("LBM_TUNE_NO_COOP", "LBM_TUNE_NO_TILE"):
        monkeypatch.delenv(v, raising=False)
    s = binding.LBM(wl)
    if inp.get("mask") is not None:
        s.set_solid_mask(inp["mask"])
    dt = np.float32 if wl["compute_dtype"] == "f32" else np.float64
    s.init_fields([np.asarray(r, dtype=dt) for r in inp["rho"]])
    for n in calls:
        if plain:
            for _ in range(n):
                s.step(1)
        else:
            s.step(n)
    assert s.hot_path == ("two_pass" if plain else "one_pass_tile"), s.hot_path
    assert s.steps_done == sum(calls)
    f = [s.get_populations(k) for k in range(s.nc)]
    macro = s.get_macroscopic()
    s.close()
    return f, macro


def d2q9(nx, ny, nc, dtype, store=None, collision="BGK", tau=1.0, periodic=(True, True, True)):
    if nc == 1:
        wl, _ = W.config1(8, dtype)
    else:
        wl, _ = W.config2(16, 8, dtype, wall=1)
    wl = dict(wl)
    wl.update(nx=nx, ny=ny, periodic=periodic, store_dtype=store or dtype, collision=collision, tau=[tau] * nc)
    if collision == "MRT":
        wl["mrt_rates"] = [W.mrt_rates("D2Q9", tau)] * nc
    return wl


def plates(nx, ny, wall):
    y = np.arange(nx * ny) // nx
    return ((y < wall) | (y >= ny - wall)).astype(np.uint8)


CASES = {
    # name: (workload, mask builder or None, density range)
    "narrower_than_the_ring": (lambda: d2q9(5, 3, 1, "f64"), None, (0.05, 0.25)),
    "one_row": (lambda: d2q9(200, 1, 1, "f64"), None, (0.05, 0.25)),
    "ragged_8x8_tiles": (lambda: d2q9(70, 37, 1, "f64", collision="MRT", tau=0.8), None, (0.05, 0.25)),
    "ragged_16x16_tiles": (lambda: d2q9(150, 93, 1, "f32"), None, (0.05, 0.25)),
    "plates_one_cell_thick": (lambda: d2q9(61, 19, 2, "f64", tau=0.9), lambda wl: plates(61, 19, 1), (0.1, 0.9)),
    "plates_32x16_tiles_mrt": (lambda: d2q9(300, 170, 2, "f32", collision="MRT", tau=1.1), lambda wl: plates(300, 170, 5), (0.1, 0.9)),
    "plates_64x16_tiles_fp16_store": (lambda: d2q9(600, 200, 2, "f32", store="f16"), lambda wl: plates(600, 200, 7), (0.1, 0.9)),
    "random_solids": (lambda: d2q9(97, 45, 2, "f64"), "random", (0.1, 0.9)),
    "closed_box": (lambda: d2q9(44, 29, 1, "f64", periodic=(False, False, True)), None, (0.05, 0.25)),
}


@pytest.mark.parametrize("name", sorted(CASES))
def test_tile_kernel_is_bit_identical_to_plain_launches(name, monkeypatch):
    mk, mask_fn, (lo, hi) = CASES[name]
    wl = mk()
    mask = None
    if mask_fn == "random":
        rng = np.random.default_rng(3)
        mask = (rng.uniform(size=wl["nx"] * wl["ny"]) < 0.18).astype(np.uint8)
    elif mask_fn is not None:
        mask = mask_fn(wl)
    inp = small_inputs(wl, 5, lo, hi, mask=mask)
    calls = (2, 37, 64)          # an even and an odd count: the ping-pong parity carries over between calls
    ft, mt = run_gpu(wl, inp, calls, monkeypatch, plain=False)
    fp, mp = run_gpu(wl, inp, calls, monkeypatch, plain=True)
    fluid = fluid_mask(inp, wl["nx"] * wl["ny"])
    for k in range(len(fp)):
        assert np.isfinite(ft[k][:, fluid]).all()
        assert np.array_equal(ft[k][:, fluid], fp[k][:, fluid]), (name, k)
    for a, b in zip(mt[0], mp[0]):   # rho incl. the virtual density of the boundary solids (refreshed by the export)
        assert np.array_equal(a, b)
    # ... and the oracle (fp16 storage: its gate is held by the plain launches in test_gpu_parity.py, to which this path is
    # bit-identical; two components at these densities leave it within 103 steps)
    if wl["store_dtype"] == "f16":
        return
    o = make_oracle(with_dtype(wl, "f64") if wl["compute_dtype"] == "f32" and wl["store_dtype"] == "f32" else wl, inp)
    o.step(sum(calls))
    fo = [o.get_populations(k) for k in range(o.nc)]
    if wl["compute_dtype"] == "f32":
        assert_parity(fo, ft, fluid, TOL32, relative=True)
    else:
        assert_parity(fo, ft, fluid, TOL64, relative=False)


def test_tile_kernel_with_velocity_inlet_and_pressure_outlet(monkeypatch):
    """Non-periodic x with a velocity face and a pressure face, plates along y: the face rules at the writing cell (R10) and
    the clamped neighbour offsets of edge cells inside the tile kernel."""
    wl = d2q9(120, 40, 2, "f64", tau=0.9, periodic=(False, True, True))
    wl["face_bc"] = {0: ("VELOCITY", (1.0, 0.03), (1e-3, 0.0, 0.0)), 1: ("PRESSURE", (0.03, 1.0), (0.0, 0.0, 0.0))}
    mask = plates(120, 40, 3)
    x = np.arange(120 * 40) % 120
    inp = dict(rho=[np.where(x < 10, 1.0, 0.03).astype(np.float64), np.where(x < 10, 0.03, 1.0).astype(np.float64)], u=None, mask=mask)
    calls = (50, 51)
    ft, _ = run_gpu(wl, inp, calls, monkeypatch, plain=False)
    fp, _ = run_gpu(wl, inp, calls, monkeypatch, plain=True)
    fluid = fluid_mask(inp, 120 * 40)
    for k in range(2):
        assert np.array_equal(ft[k][:, fluid], fp[k][:, fluid])
    o = make_oracle(wl, inp)
    o.step(sum(calls))
    assert_parity([o.get_populations(k) for k in range(2)], ft, fluid, TOL64, relative=False)
