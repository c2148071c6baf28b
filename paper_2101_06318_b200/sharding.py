"""Host-side logic for running the SDM coalescence step on several GPUs (one process per GPU).

Collisions happen only between super-droplets of the same cell, so a grid workload
shards by CONTIGUOUS CELL RANGES with no exchange inside a coalescence step: every rank owns a
``libsdm`` handle for its cells and steps it independently.  The only collective on the path is the
all-reduce of the three global moments, 24 bytes per rank.  Single-cell box workloads
do not shard (one global permutation): they run as independent replicas.

A sharded run reproduces the unsharded one exactly: every shard uses the SAME Philox seed and tells its handle
the global storage index of its first droplet (``sdm_set_index_base``); the stable compaction shifts later
shards, so after a removal the bases are re-derived from the survivor counts (``rebase``: an exclusive scan of
one integer per rank).  Replicas of a single-cell box (independent realisations) use ``shard_seed`` instead.

Nothing here touches the method's arithmetic; it cuts arrays, scans counts and reduces three numbers.
(DESIGN.md section 9.)
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

_MASK64 = (1 << 64) - 1


@dataclass
class CellRange:
    rank: int
    cell_lo: int        # first cell of the shard
    cell_hi: int        # one past the last cell
    sd_lo: int          # first super-droplet (cell-contiguous storage)
    sd_hi: int


def partition_cells(counts, world: int) -> list[CellRange]:
    """Cuts ``len(counts)`` cells into ``world`` contiguous ranges with (nearly) equal droplet counts:
    boundary r is the first cell whose droplet prefix reaches r/world of the total.  Every cell goes to
    exactly one rank; ranges may be empty when there are fewer cells than ranks."""
    counts = np.asarray(counts, dtype=np.int64)
    if world < 1:
        raise ValueError("world must be >= 1")
    n_cell = int(counts.shape[0])
    prefix = np.concatenate([[0], np.cumsum(counts)])
    total = int(prefix[-1])
    bounds = [0]
    for r in range(1, world):
        target = (total * r + world - 1) // world
        b = int(np.searchsorted(prefix, target, side="left"))
        bounds.append(min(max(b, bounds[-1]), n_cell))
    bounds.append(n_cell)
    return [CellRange(r, bounds[r], bounds[r + 1], int(prefix[bounds[r]]), int(prefix[bounds[r + 1]]))
            for r in range(world)]


def shard_seed(seed: int, rank: int) -> int:
    """Philox key of a REPLICA (independent realisations of a box; NOT for shards of one state, which
    share the seed and differ in their index base): the simulation seed advanced by ``rank`` odd constants (a Weyl
    sequence: distinct for distinct ranks, rank 0 keeps the seed itself)."""
    return (int(seed) + int(rank) * 0x9E3779B97F4A7C15) & _MASK64


def index_bases(counts) -> list[int]:
    """Global storage index of every shard's first droplet: the exclusive scan of the shards' droplet counts."""
    out, run = [], 0
    for c in counts:
        out.append(run)
        run += int(c)
    return out


def rebase(n_local: int, rank: int, world: int, group=None) -> int:
    """This rank's index base after a compaction: all-gather of the survivor counts (one int64 per rank), exclusive
    scan.  With no initialised process group: 0 (a single shard)."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or world == 1:
        return 0
    mine = torch.tensor([int(n_local)], dtype=torch.int64)
    if dist.get_backend(group) == "nccl":
        mine = mine.cuda()
    allc = [torch.zeros_like(mine) for _ in range(world)]
    dist.all_gather(allc, mine, group=group)
    return index_bases([int(t.item()) for t in allc])[rank]


def shard_state(xi, v, cell_id, n_cell: int, rank: int, world: int):
    """Returns (xi, v, local_cell_id, n_cell_local, CellRange) of this rank's cells.  Storage that is
    not cell-contiguous is first put in cell order by a STABLE sort, which keeps the relative storage
    order inside every cell (the order the RNG counter and the tie rule see)."""
    xi, v, cell_id = np.asarray(xi), np.asarray(v), np.asarray(cell_id)
    if cell_id.size and np.any(np.diff(cell_id) < 0):
        order = np.argsort(cell_id, kind="stable")
        xi, v, cell_id = xi[order], v[order], cell_id[order]
    counts = np.bincount(cell_id, minlength=n_cell)
    cr = partition_cells(counts, world)[rank]
    sl = slice(cr.sd_lo, cr.sd_hi)
    local_cell = (cell_id[sl] - cr.cell_lo).astype(np.int32)
    return (np.ascontiguousarray(xi[sl]), np.ascontiguousarray(v[sl]), np.ascontiguousarray(local_cell),
            max(cr.cell_hi - cr.cell_lo, 1), cr)


def allreduce_moments(m0, m1, m2, group=None):
    """Global moments from per-shard moments: M0 is summed exactly in int64, M1 and M2 in fp64.
    Arguments are torch tensors (any device the process group supports) or Python numbers; returns
    (int, float, float).  With no initialised process group the local values are returned."""
    import torch
    import torch.distributed as dist

    def _t(x, dtype):
        return x.detach().clone().reshape(-1)[:1].to(dtype) if torch.is_tensor(x) else torch.tensor([x], dtype=dtype)

    t0, t12 = _t(m0, torch.int64), torch.cat([_t(m1, torch.float64), _t(m2, torch.float64).to(_t(m1, torch.float64).device)])
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(t0, op=dist.ReduceOp.SUM, group=group)
        dist.all_reduce(t12, op=dist.ReduceOp.SUM, group=group)
    return int(t0.item()), float(t12[0].item()), float(t12[1].item())


class DeviceMoments:
    """Global moments of a sharded state WITHOUT leaving the device (the step stays asynchronous): the three local
    moments live in one 24-byte buffer that ``sdm_coalescence_step_moments`` writes; ``reduce()`` all-gathers the raw
    buffers (one collective, dtype-agnostic, NCCL or gloo) and sums them -- M0 exactly in int64, M1 and M2 in fp64."""

    def __init__(self, device, world: int, group=None):
        import torch

        self.torch, self.world, self.group = torch, int(world), group
        self.buf = torch.zeros(3, dtype=torch.int64, device=device)
        self.out = (self.buf[0:1], self.buf[1:2].view(torch.float64), self.buf[2:3].view(torch.float64))
        self.gathered = torch.zeros((self.world, 3), dtype=torch.int64, device=device)
        self.m0 = torch.zeros(1, dtype=torch.int64, device=device)
        self.m12 = torch.zeros(2, dtype=torch.float64, device=device)

    def reduce(self):
        """Enqueues the collective and the two sums on the current stream; returns (m0, m12) device tensors."""
        import torch.distributed as dist

        t = self.torch
        if self.world > 1 and dist.is_available() and dist.is_initialized():
            dist.all_gather_into_tensor(self.gathered.view(-1), self.buf, group=self.group)
        else:
            self.gathered[0].copy_(self.buf)
        t.sum(self.gathered[:, 0], dim=0, keepdim=True, out=self.m0)
        t.sum(self.gathered[:, 1:].view(t.float64), dim=0, out=self.m12)
        return self.m0, self.m12

    def values(self):
        """(M0 int, M1 float, M2 float) on the host (synchronises)."""
        return int(self.m0.item()), float(self.m12[0].item()), float(self.m12[1].item())


def max_over_ranks(value: float, device=None, group=None) -> float:
    """Timing rule of bench.py: a multi-GPU duration is the maximum over ranks."""
    import torch
    import torch.distributed as dist

    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())
