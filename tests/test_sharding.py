"""Multi-GPU host logic on CPU: two `gloo` ranks shard a grid workload by contiguous cell ranges, step
their shards independently (the CPU oracle stands in for the device: the data path needs no collective)
and all-reduce the three global moments.  DESIGN.md section 9."""
import os
import socket

import numpy as np
import pytest

import oracle
import workloads
from paper_2101_06318_b200 import sharding

torch = pytest.importorskip("torch")


def test_partition_covers_every_cell_once_and_balances_droplets():
    rng = np.random.default_rng(0)
    counts = rng.poisson(64, 1000)
    for world in (1, 2, 3, 8):
        parts = sharding.partition_cells(counts, world)
        assert parts[0].cell_lo == 0 and parts[-1].cell_hi == 1000
        for a, b in zip(parts, parts[1:]):
            assert a.cell_hi == b.cell_lo and a.sd_hi == b.sd_lo
        sizes = [p.sd_hi - p.sd_lo for p in parts]
        assert sum(sizes) == counts.sum()
        assert max(sizes) - min(sizes) <= 2 * counts.max()
    # fewer cells than ranks, empty cells, empty state
    parts = sharding.partition_cells([5, 0, 7], 5)
    assert [(p.cell_lo, p.cell_hi) for p in parts][-1][1] == 3
    assert sum(p.sd_hi - p.sd_lo for p in parts) == 12
    assert all(p.sd_hi == 0 for p in sharding.partition_cells([0, 0], 2))


def test_index_bases_are_the_exclusive_scan_of_the_counts():
    assert sharding.index_bases([5, 0, 7, 3]) == [0, 5, 5, 12]
    assert sharding.index_bases([]) == [] and sharding.rebase(10, 0, 1) == 0


def test_shard_seeds_are_distinct_and_rank0_keeps_the_seed():
    seeds = {sharding.shard_seed(7, r) for r in range(64)}
    assert len(seeds) == 64 and sharding.shard_seed(7, 0) == 7
    assert all(0 <= s < 2 ** 64 for s in seeds)


def test_shard_state_of_shuffled_storage_keeps_in_cell_order():
    w = workloads.grid_small_multiplicity(8, 8, 10, shuffled=True, seed=3)
    seen = 0
    for rank in range(3):
        xi, v, cell, n_local, cr = sharding.shard_state(w.xi, w.v, w.cell_id, w.n_cell, rank, 3)
        assert np.all(np.diff(cell) >= 0) and (cell.size == 0 or cell.max() < n_local)
        for c in range(cr.cell_lo, cr.cell_hi):
            assert np.array_equal(xi[cell == c - cr.cell_lo], w.xi[w.cell_id == c])      # stable inside a cell
        seen += xi.size
    assert seen == w.n_sd


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank, world, port, ret):
    import torch.distributed as dist

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = workloads.grid_small_multiplicity(12, 12, 24, seed=5)
        xi, v, cell, n_local, _ = sharding.shard_state(w.xi, w.v, w.cell_id, w.n_cell, rank, world)
        for step in range(6):
            xi, v, cell = oracle.remove_zero(xi, v, cell)
            base = sharding.rebase(len(xi), rank, world)          # all-gather of the survivor counts
            sid = base + np.arange(len(xi), dtype=np.int64)       # what sdm_set_index_base tells the device
            oracle.step(xi, v, cell, n_local, w.dt, w.dV, w.kernel, w.kparam, w.seed, step, sid=sid)
        m0, m1, m2 = oracle.moments(xi, v)
        ret[("state", rank)] = (xi.copy(), v.copy())
        g = sharding.allreduce_moments(torch.tensor([m0]), torch.tensor([m1], dtype=torch.float64),
                                       torch.tensor([m2], dtype=torch.float64))
        t = sharding.max_over_ranks(1.0 + rank)
        dm = sharding.DeviceMoments("cpu", world)                 # the device-side variant bench.py uses (here on gloo)
        dm.out[0][0], dm.out[1][0], dm.out[2][0] = m0, m1, m2
        dm.reduce()
        assert dm.values() == g
        ret[rank] = (m0, m1, m2, g, t)
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_step_their_shards_and_allreduce_moments():
    import torch.multiprocessing as mp

    world, port = 2, _free_port()
    with mp.Manager() as mgr:
        ret = mgr.dict()
        mp.spawn(_rank_main, args=(world, port, ret), nprocs=world, join=True)
        out = dict(ret)
    states = {k[1]: out.pop(k) for k in list(out) if isinstance(k, tuple)}
    assert set(out) == {0, 1}
    m0 = sum(out[r][0] for r in out)
    m1 = sum(out[r][1] for r in out)
    m2 = sum(out[r][2] for r in out)
    # the sharded run IS the unsharded one: same seed, global storage indices re-derived after every removal
    w = workloads.grid_small_multiplicity(12, 12, 24, seed=5)
    xi, v, cell = w.xi.copy(), w.v.copy(), w.cell_id.copy()
    for step in range(6):
        xi, v, cell = oracle.remove_zero(xi, v, cell)
        oracle.step(xi, v, cell, w.n_cell, w.dt, w.dV, w.kernel, w.kparam, w.seed, step)
    assert np.array_equal(np.concatenate([states[0][0], states[1][0]]), xi)
    assert np.array_equal(np.concatenate([states[0][1], states[1][1]]), v)
    assert len(xi) < w.n_sd                                       # removals shifted the second shard's base
    for r in out:
        g0, g1, g2 = out[r][3]
        assert g0 == m0 and abs(g1 - m1) <= 1e-12 * m1 and abs(g2 - m2) <= 1e-12 * m2
        assert out[r][4] == 2.0                                   # max over ranks of (1, 2)
    # water is conserved across the sharded run (Golovin C6 workload: sum xi v is invariant)
    w = workloads.grid_small_multiplicity(12, 12, 24, seed=5)
    assert abs(m1 - oracle.moments(w.xi, w.v)[1]) <= 1e-12 * m1
    assert m0 < int(w.xi.sum())                                   # collisions happened on both shards
