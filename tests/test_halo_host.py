"""Host logic of the slab decomposition (paper_2506_17713_b200/halo.py), no GPU: the partition, the neighbours, and the
exchange protocol over gloo with world_size 2 -- each rank steps ITS slab with the oracle, exchanges `width` ghost layers
before every step through halo.exchange, and the owned layers must equal the undecomposed oracle run bit for bit (the
same cells see the same neighbour values).  The GPU side of the same protocol is tests/test_gpu_halo.py."""
import os
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))
from paper_2506_17713_b200 import halo  # noqa: E402
from paper_2506_17713_b200 import workloads as W  # noqa: E402


def test_slabs_partition_the_axis_and_name_their_neighbours():
    for n_last, world, width in [(64, 2, 2), (65, 4, 2), (30, 3, 3), (8, 1, 2)]:
        slabs = [halo.Slab(n_last, world, r, width) for r in range(world)]
        owned = [l for s in slabs for l in range(s.lo, s.hi)]
        assert owned == list(range(n_last))                       # disjoint, complete, in rank order
        assert max(s.hi - s.lo for s in slabs) - min(s.hi - s.lo for s in slabs) <= 1
        for s in slabs:
            assert s.n_local == s.hi - s.lo + 2 * width
            assert s.neighbour(0) == (s.rank - 1) % world and s.neighbour(1) == (s.rank + 1) % world
            g = s.global_layers()
            assert len(g) == s.n_local and g[s.interior()] == list(range(s.lo, s.hi))
            assert g[0] == (s.lo - width) % n_last and g[-1] == (s.hi + width - 1) % n_last
    ends = [halo.Slab(40, 4, r, 2, periodic=False) for r in range(4)]
    assert ends[0].neighbour(0) is None and ends[3].neighbour(1) is None and ends[1].neighbour(0) == 0
    with pytest.raises(ValueError):
        halo.Slab(6, 4, 3, 2)                                     # a slab thinner than the halo


class OracleSlab:
    """The oracle on one slab, with the calls halo.exchange needs.  Its state is f(x, t) after streaming, so the
    ghost layers carry the neighbours' f(x, t); the widths are those of include/lbm.h."""

    def __init__(self, wl, inp, slab, layer_cells):
        import torch
        from oracle import lbm_oracle as O
        self.torch, self.slab, self.lc = torch, slab, layer_cells
        g = np.asarray(slab.global_layers())
        lwl = dict(wl)
        last = "nz" if wl["lattice"] == "D3Q19" else "ny"
        lwl[last] = slab.n_local
        take = lambda a: np.ascontiguousarray(np.asarray(a).reshape(-1, layer_cells)[g]).reshape(-1)
        self.sim = O.Oracle(lwl)
        if inp.get("mask") is not None:
            self.sim.set_solid_mask(take(inp["mask"]))
        self.sim.init_fields([take(r) for r in inp["rho"]])
        self.nc, self.q = self.sim.nc, self.sim.q

    def _layers(self, side, export):
        w, n = self.slab.width, self.slab.n_local
        if export:
            return slice(w, 2 * w) if side == 0 else slice(n - 2 * w, n - w)
        return slice(0, w) if side == 0 else slice(n - w, n)

    def halo_bytes(self, width):
        return self.nc * self.q * width * self.lc * 8

    def export_halo(self, side, width):
        f = np.stack([self.sim.get_populations(k) for k in range(self.nc)])          # [nc][q][N]
        f = f.reshape(self.nc, self.q, self.slab.n_local, self.lc)[:, :, self._layers(side, True)]
        return self.torch.from_numpy(np.ascontiguousarray(f).reshape(-1).view(np.uint8).copy())

    def import_halo(self, side, width, buf):
        g = buf.numpy().view(np.float64).reshape(self.nc, self.q, width, self.lc)
        for k in range(self.nc):
            f = self.sim.get_populations(k).reshape(self.q, self.slab.n_local, self.lc)
            f[:, self._layers(side, False)] = g[k]
            self.sim.set_populations(k, f.reshape(self.q, -1))

    def owned(self):
        f = np.stack([self.sim.get_populations(k) for k in range(self.nc)])
        return f.reshape(self.nc, self.q, self.slab.n_local, self.lc)[:, :, self.slab.interior()]


def _case(name):
    if name == "plain":       # config 1 physics on a 24 x 36 box, slabs along y, width 2
        wl, _ = W.config1(16, "f64")
        wl.update(nx=24, ny=36)
        rng = np.random.default_rng(3)
        rho = np.where(rng.random(24 * 36) < 0.3, 0.30, 0.05) + rng.uniform(-1e-3, 1e-3, 24 * 36)
        return wl, dict(rho=[rho], mask=None), halo.HALO_WIDTH_FLUID, 24
    # two components and a solid obstacle with virtual-density wetting that straddles the cut: width 3
    wl, _ = W.config2(16, 16, "f64")
    wl.update(nx=20, ny=40)
    rng = np.random.default_rng(4)
    y, x = np.divmod(np.arange(20 * 40), 20)
    mask = ((np.abs(y - 20) <= 2) & (x > 4) & (x < 14)).astype(np.uint8) | ((y < 2) & (x < 6)).astype(np.uint8)
    a = np.where(x < 10, 1.0, 0.03) + rng.uniform(-1e-3, 1e-3, x.size)
    b = np.where(x < 10, 0.03, 1.0) + rng.uniform(-1e-3, 1e-3, x.size)
    return wl, dict(rho=[a, b], mask=mask), halo.HALO_WIDTH_WETTING, 20


def _reference(wl, inp, steps, lc):
    from oracle import lbm_oracle as O
    ref = O.Oracle(wl)
    if inp["mask"] is not None:
        ref.set_solid_mask(inp["mask"])
    ref.init_fields(inp["rho"])
    ref.step(steps)
    return np.stack([ref.get_populations(k) for k in range(ref.nc)]).reshape(ref.nc, ref.q, wl["ny"], lc)


def _worker(rank, world, port, case, steps, out):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="1")
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl, inp, width, lc = _case(case)
    slab = halo.Slab(wl["ny"], world, rank, width)
    sim = OracleSlab(wl, inp, slab, lc)
    for _ in range(steps):
        halo.exchange(sim, slab, dist)
        sim.sim.step(1)
    dist.barrier()
    out.put((rank, slab.lo, slab.hi, sim.owned()))
    dist.destroy_process_group()


@pytest.mark.parametrize("case", ["plain", "wetting"])
def test_two_slabs_over_gloo_equal_the_undecomposed_run(case):
    import torch.multiprocessing as mp
    steps = 12
    wl, inp, width, lc = _case(case)
    want = _reference(wl, inp, steps, lc)
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, case, steps, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = [out.get(timeout=240) for _ in range(2)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, lo, hi, f in got:
        assert f.shape == want[:, :, lo:hi].shape
        fluid = np.ones(f.shape, bool)
        if inp["mask"] is not None:                        # solid cells hold no state
            fluid &= (inp["mask"].reshape(wl["ny"], lc)[lo:hi] == 0)[None, None]
        assert np.array_equal(f[fluid], want[:, :, lo:hi][fluid]), f"rank {rank}: slab differs from the undecomposed run"


@pytest.mark.parametrize("case", ["plain", "wetting"])
def test_three_slabs_in_one_process_and_the_width_is_necessary(case):
    """halo.exchange_local over three slabs; with one ghost layer less than include/lbm.h asks for, the owned layers
    must NOT reproduce the undecomposed run (otherwise the equality above would say nothing about the width)."""
    steps = 10
    wl, inp, width, lc = _case(case)
    want = _reference(wl, inp, steps, lc)
    fluid_all = np.ones(wl["ny"] * lc, bool) if inp["mask"] is None else inp["mask"] == 0
    for w, must_match in [(width, True), (width - 1, False)]:
        slabs = [halo.Slab(wl["ny"], 3, r, w) for r in range(3)]
        sims = [OracleSlab(wl, inp, s, lc) for s in slabs]
        for _ in range(steps):
            halo.exchange_local(sims, slabs)
            for s in sims:
                s.sim.step(1)
        same = True
        for s, sl in zip(sims, slabs):
            fl = np.broadcast_to(fluid_all.reshape(wl["ny"], lc)[sl.lo:sl.hi][None, None], s.owned().shape)
            same &= np.array_equal(s.owned()[fl], want[:, :, sl.lo:sl.hi][fl])
        assert same == must_match, (w, same)
