"""Slab decomposition of the domain along its last axis and the halo exchange between the slabs.

The path's only real exchange step: the stored populations of `width` layers on either side of a slab
(include/lbm.h, lbm_export_halo / lbm_import_halo).  One process per GPU; the messages travel as point-to-point
torch.distributed operations (NCCL over NVLink between GPUs; gloo in the CPU tests), batched so that both directions
are in flight at once.  This module holds host logic only: which layers a rank owns, who its neighbours are, and the
order of the four messages.  Anything with `halo_bytes(width)`, `export_halo(side, width)`, `import_halo(side, width, buf)`
can be exchanged (binding.LBM on the GPU; the tests drive the same code with a CPU stepper over gloo).
"""
from __future__ import annotations

from dataclasses import dataclass

HALO_WIDTH_FLUID = 2      # plain Shan-Chen step: psi one layer out, from populations pulled one layer further
HALO_WIDTH_WETTING = 3    # + virtual density of solid cells in the first ghost layer (Eq. 17 averages one layer further)


@dataclass(frozen=True)
class Slab:
    """Rank `rank` of `world` owns layers [lo, hi) of the `n_last` global layers; its handle is built with
    `n_local = hi - lo + 2 * width` layers: `width` ghost layers, the owned ones, `width` ghost layers."""
    n_last: int
    world: int
    rank: int
    width: int
    periodic: bool = True

    def __post_init__(self):
        if not (0 <= self.rank < self.world):
            raise ValueError("rank outside the world")
        if self.width < 1:
            raise ValueError("width >= 1")
        if self.hi - self.lo < self.width:
            raise ValueError("a slab must own at least `width` layers")

    @property
    def lo(self) -> int:
        base, rem = divmod(self.n_last, self.world)
        return self.rank * base + min(self.rank, rem)

    @property
    def hi(self) -> int:
        base, rem = divmod(self.n_last, self.world)
        return self.lo + base + (1 if self.rank < rem else 0)

    @property
    def n_local(self) -> int:
        return self.hi - self.lo + 2 * self.width

    def neighbour(self, side: int):
        """Rank on the low (0) / high (1) side, or None at a non-periodic end."""
        r = self.rank + (1 if side else -1)
        if 0 <= r < self.world:
            return r
        return r % self.world if self.periodic else None

    def global_layers(self):
        """Global layer index of every local layer (ghost layers wrap around a periodic domain; at a non-periodic
        end they repeat the edge layer -- the caller's boundary treatment owns those)."""
        out = []
        for l in range(self.lo - self.width, self.hi + self.width):
            out.append(l % self.n_last if self.periodic else min(max(l, 0), self.n_last - 1))
        return out

    def interior(self) -> slice:
        return slice(self.width, self.width + self.hi - self.lo)


def exchange_local(sims, slabs) -> None:
    """Halo exchange between handles that live in ONE process (several slabs on one GPU, or a test)."""
    by_rank = {s.rank: (sim, s) for sim, s in zip(sims, slabs)}
    packed = {}
    for r, (sim, s) in by_rank.items():
        for side in (0, 1):
            if s.neighbour(side) is not None:
                packed[(r, side)] = sim.export_halo(side, s.width)
    for r, (sim, s) in by_rank.items():
        for side in (0, 1):
            nb = s.neighbour(side)
            if nb is not None:
                sim.import_halo(side, s.width, packed[(nb, 1 - side)])   # my low ghost layers = their high interior edge


def exchange(sim, slab: Slab, dist, recv_bufs=None, group=None) -> None:
    """Halo exchange of this rank's handle with its neighbours (one process per GPU).

    `dist` is torch.distributed (initialised).  Up to four messages, all posted before any is waited for; a rank that is
    its own neighbour on both sides (world == 1, periodic) copies locally.  `recv_bufs`: optional pair of preallocated
    receive tensors (like the ones export_halo returns)."""
    w = slab.width
    if slab.world == 1:
        if slab.periodic:
            lo, hi = sim.export_halo(0, w), sim.export_halo(1, w)
            sim.import_halo(0, w, hi)
            sim.import_halo(1, w, lo)
        return
    # Receives are posted low side first, sends high side first: my high-side export is the neighbour's low-side import,
    # so between two ranks that are each other's neighbour on BOTH sides (world == 2) the k-th send meets the k-th
    # receive -- NCCL matches the messages of a pair in posting order and ignores tags; gloo also gets the tag.
    sends = {side: sim.export_halo(side, w) for side in (0, 1) if slab.neighbour(side) is not None}
    ops, recvs = [], {}
    for side in (0, 1):
        if side not in sends:
            continue
        recv = recv_bufs[side] if recv_bufs is not None else sends[side].new_empty(sends[side].shape)
        recvs[side] = recv
        ops.append(dist.P2POp(dist.irecv, recv, slab.neighbour(side), group=group, tag=side))
    for side in (1, 0):
        if side in sends:
            ops.append(dist.P2POp(dist.isend, sends[side], slab.neighbour(side), group=group, tag=1 - side))
    for req in dist.batch_isend_irecv(ops):
        req.wait()
    for side, recv in recvs.items():
        sim.import_halo(side, w, recv)
