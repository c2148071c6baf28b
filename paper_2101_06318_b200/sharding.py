"""Host-side logic for running the SDM coalescence step on several GPUs (one process per GPU).

Collisions happen only between super-droplets of the same cell, so a grid workload
shards by CONTIGUOUS CELL RANGES with no exchange inside a coalescence step: every rank owns a
``libsdm`` handle for its cells and steps it independently.  The only collective on the path is the
all-reduce of the three global moments, 24 bytes per rank.  Single-cell box workloads
do not shard (one global permutation): they run as independent replicas.

Nothing here touches the method's arithmetic; it cuts arrays, derives per-shard seeds and reduces three
numbers.  (DESIGN.md section 9.)
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
    """Philox key of a shard: shards must not reuse one another's random stream (their storage indices
    all start at 0), so the 64-bit key is the simulation seed advanced by ``rank`` odd constants
    (a Weyl sequence: distinct for distinct ranks, rank 0 keeps the seed itself)."""
    return (int(seed) + int(rank) * 0x9E3779B97F4A7C15) & _MASK64


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


def max_over_ranks(value: float, device=None, group=None) -> float:
    """Timing rule of bench.py: a multi-GPU duration is the maximum over ranks."""
    import torch
    import torch.distributed as dist

    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())
