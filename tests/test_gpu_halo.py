"""Slab decomposition on the GPU (lbm_export_halo / lbm_import_halo, include/lbm.h): several handles on one GPU, each
a slab of the last axis with ghost layers, exchanging before every step through halo.exchange_local -- their owned layers
must equal the undecomposed run BIT FOR BIT (every owned cell sees the same neighbour values and the kernels do the same
arithmetic whatever the domain size), and the undecomposed run is the one the other tests hold against the oracle.
The protocol over torch.distributed is covered on the CPU (tests/test_halo_host.py, gloo, world_size 2)."""
import numpy as np
import pytest

from paper_2506_17713_b200 import halo
from paper_2506_17713_b200 import workloads as W
from test_gpu_parity import make_gpu, small_inputs

pytestmark = pytest.mark.gpu


def run_slabs(wl, inp, steps, world, width):
    """-> (owned populations per slab [nc][q][layers][cells], populations of the undecomposed run [nc][q][n_last][cells])"""
    d3 = wl["lattice"] == "D3Q19"
    last = "nz" if d3 else "ny"
    lc = wl["nx"] * wl["ny"] if d3 else wl["nx"]
    ref = make_gpu(wl, inp)
    ref.step(steps)
    want = np.stack([ref.get_populations(k) for k in range(wl["n_components"])]).reshape(wl["n_components"], ref.q, wl[last], lc)
    slabs = [halo.Slab(wl[last], world, r, width) for r in range(world)]
    sims = []
    for s in slabs:
        g = np.asarray(s.global_layers())
        take = lambda a: np.ascontiguousarray(np.asarray(a).reshape(-1, lc)[g]).reshape(-1)
        lwl = dict(wl)
        lwl[last] = s.n_local
        linp = dict(rho=[take(r) for r in inp["rho"]], u=None, mask=None if inp.get("mask") is None else take(inp["mask"]))
        sims.append(make_gpu(lwl, linp))
    for _ in range(steps):
        halo.exchange_local(sims, slabs)
        for sim in sims:
            sim.step(1)
    halo.exchange_local(sims, slabs)      # exports pull across the cut too (include/lbm.h): exchange before reading
    got = []
    for sim, s in zip(sims, slabs):
        f = np.stack([sim.get_populations(k) for k in range(wl["n_components"])])
        got.append(f.reshape(wl["n_components"], sim.q, s.n_local, lc)[:, :, s.interior()])
    return got, want, slabs, sims


@pytest.mark.parametrize("path,hot", [("one_pass", "one_pass_eq"), ("two_pass", "two_pass")])
@pytest.mark.parametrize("dtype,store", [("f64", "f64"), ("f32", "f32"), ("f32", "f16")])
def test_d3q19_two_and_three_slabs_equal_the_whole_domain(dtype, store, path, hot):
    wl, _ = W.config5(16, dtype, store)
    wl.update(nx=128, ny=16, nz=36, path=path)
    inp = small_inputs(wl, 7, 0.05, 0.3)
    for world in (2, 3):
        got, want, slabs, sims = run_slabs(wl, inp, 8, world, halo.HALO_WIDTH_FLUID)
        assert {s.hot_path for s in sims} == {hot}
        for f, s in zip(got, slabs):
            d = np.abs(f - want[:, :, s.lo:s.hi]).max()
            assert np.array_equal(f, want[:, :, s.lo:s.hi]), f"slab {s.rank} of {world}: max |diff| {d:.3e}"


def test_d2q9_two_components_wetting_obstacle_across_the_cut():
    """Two components, plates and an obstacle with virtual-density wetting straddling the cut: width 3."""
    wl, _ = W.config2(16, 16, "f64")
    wl.update(nx=32, ny=48)
    y, x = np.divmod(np.arange(32 * 48), 32)
    mask = ((np.abs(y - 24) <= 2) & (x > 6) & (x < 20)).astype(np.uint8) | ((y < 2) & (x < 9)).astype(np.uint8)
    rng = np.random.default_rng(11)
    a = np.where(x < 16, 1.0, 0.03) + rng.uniform(-1e-3, 1e-3, x.size)
    b = np.where(x < 16, 0.03, 1.0) + rng.uniform(-1e-3, 1e-3, x.size)
    inp = dict(rho=[a, b], u=None, mask=mask)
    fluid = (mask == 0).reshape(48, 32)
    got, want, slabs, _ = run_slabs(wl, inp, 12, 2, halo.HALO_WIDTH_WETTING)
    for f, s in zip(got, slabs):
        fl = np.broadcast_to(fluid[s.lo:s.hi][None, None], f.shape)
        assert np.array_equal(f[fl], want[:, :, s.lo:s.hi][fl])
    # one ghost layer less does not reproduce it (the equality above depends on the width)
    got, want, slabs, _ = run_slabs(wl, inp, 12, 2, halo.HALO_WIDTH_WETTING - 1)
    assert not all(np.array_equal(f[np.broadcast_to(fluid[s.lo:s.hi][None, None], f.shape)],
                                  want[:, :, s.lo:s.hi][np.broadcast_to(fluid[s.lo:s.hi][None, None], f.shape)])
                   for f, s in zip(got, slabs))


def test_halo_buffer_layout_and_errors():
    """The packed buffer is [component][direction][layer][cells] of the stored populations; bad arguments are refused."""
    import torch
    from paper_2506_17713_b200 import binding
    wl, _ = W.config5(16, "f32")
    wl.update(nx=8, ny=4, nz=12, path="two_pass")
    inp = small_inputs(wl, 5)
    g = make_gpu(wl, inp)
    assert g.halo_bytes(2) == 19 * 2 * 8 * 4 * 4
    lo = g.export_halo(0, 2).view(torch.float32).reshape(19, 2, 32).cpu().numpy()
    hi = g.export_halo(1, 2).view(torch.float32).reshape(19, 2, 32).cpu().numpy()
    # the stored value of direction i at cell x is the one the cell x + e_i pulls (R14), so right after lbm_init_fields the
    # packed layers are the exported (post-stream) populations shifted back by e_i
    e, _, _ = binding.get_lattice("D3Q19")
    pops = g.get_populations(0, dtype=np.float32).reshape(19, 12, 4, 8)
    for i in range(19):
        back = np.roll(pops[i], shift=(-e[i][2], -e[i][1], -e[i][0]), axis=(0, 1, 2))
        assert np.array_equal(lo[i], back[2:4].reshape(2, 32)) and np.array_equal(hi[i], back[8:10].reshape(2, 32))
    # an import into the ghost layers leaves the interior edge layers as they were
    g.import_halo(1, 2, torch.from_numpy(lo).cuda().view(torch.uint8).reshape(-1))
    assert np.array_equal(g.export_halo(1, 2).view(torch.float32).reshape(19, 2, 32).cpu().numpy(), hi)
    g.import_halo(0, 2, torch.from_numpy(hi).cuda().view(torch.uint8).reshape(-1))
    assert np.array_equal(g.export_halo(0, 2).view(torch.float32).reshape(19, 2, 32).cpu().numpy(), lo)
    for bad in [lambda: g.export_halo(2, 2), lambda: g.halo_bytes(0), lambda: g.halo_bytes(5)]:
        with pytest.raises(binding.LBMError):
            bad()
    g3 = make_gpu(dict(wl, periodic=(True, True, False)), inp)
    with pytest.raises(binding.LBMError):
        g3.halo_bytes(2)
