"""Cell-range sharding on the device: shards of ONE state in separate libsdm handles -- same
Philox seed, global storage indices through sdm_set_index_base, bases re-derived from the survivor counts after every
removal -- reproduce the oracle's UNSHARDED run bit for bit: concatenated xi and v, and idx + base.  (One GPU runs
the shards one after the other: there is no exchange inside a step, so nothing waits on anything.)"""
import numpy as np
import pytest

import oracle
import workloads
from paper_2101_06318_b200 import sharding

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def sdm_mod():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2101_06318_b200 as m
    m.load_library()
    return m


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _sharded_run(sdm_mod, w, world, steps, options=(), expect_modes=None):
    shards = []
    for rank in range(world):
        xi, v, cell, n_local, cr = sharding.shard_state(w.xi, w.v, w.cell_id, w.n_cell, rank, world)
        s = sdm_mod.SDM(max(len(xi), 1), n_local)
        for k, val in options:
            s.set_option(k, val)
        s.set_state(_dev(xi), _dev(v), _dev(cell))
        shards.append((s, cr))
    if expect_modes is not None:
        assert [s.counters()["mode"] for s, _ in shards] == expect_modes
    # the oracle steps the WHOLE state (cell-contiguous order, which is what shard_state cuts)
    order = np.argsort(w.cell_id, kind="stable")
    xi, v, cell = w.xi[order].copy(), w.v[order].copy(), w.cell_id[order].copy()
    events = 0
    for step in range(steps):
        xi, v, cell = oracle.remove_zero(xi, v, cell)
        counts = [s.remove_zero() for s, _ in shards]
        assert sum(counts) == len(xi)
        bases = sharding.index_bases(counts)
        for (s, _), b in zip(shards, bases):
            s.set_index_base(b)
        idx, cs, nev = oracle.step(xi, v, cell, w.n_cell, w.dt, w.dV, w.kernel, w.kparam, w.seed, step)
        events += nev
        gx, gv, gi = [], [], []
        for (s, cr), b, n in zip(shards, bases, counts):
            s.coalescence_step(w.dt, w.dV, w.kernel, w.kparam, w.seed, step)
            sx, sv, _ = s.get_state()
            gx.append(sx.cpu().numpy()), gv.append(sv.cpu().numpy())
            gi.append(s.get_permutation(n)[0].cpu().numpy().astype(np.int64) + b)
        assert np.array_equal(np.concatenate(gx), xi), f"xi differs at step {step}"
        assert np.array_equal(np.concatenate(gv), v), f"v differs at step {step}"
        assert np.array_equal(np.concatenate(gi), idx), f"idx + base differs at step {step}"
    assert sum(s.counters()["events"] for s, _ in shards) == events
    m = [s.moments_host() for s, _ in shards]
    o = oracle.moments(xi, v)
    assert sum(a[0] for a in m) == o[0] and abs(sum(a[1] for a in m) - o[1]) <= 1e-12 * o[1]
    for s, _ in shards:
        s.close()
    return events, len(xi)


@pytest.mark.parametrize("world", [2, 3])
def test_shards_of_a_small_multiplicity_grid_fused_path(sdm_mod, world):
    w = workloads.grid_small_multiplicity(24, 24, 32, seed=8)            # droplets vanish every step: bases move
    events, n_end = _sharded_run(sdm_mod, w, world, 20, expect_modes=[1] * world)
    assert events > 5000 and n_end < w.n_sd - 1000


def test_shards_of_a_poisson_grid_general_path_and_shuffled_storage(sdm_mod):
    w = workloads.grid_poisson(24, 24, 64.0, shuffled=True, seed=3)       # shard_state puts storage in cell order first
    w.kparam = 1500.0 * 4000.0
    events, _ = _sharded_run(sdm_mod, w, 2, 8, options=[(sdm_mod.OPT_FORCE_GENERAL, 1)], expect_modes=[0, 0])
    assert events > 50


def test_shards_of_full_cells_counting_sort_kernel(sdm_mod):
    w = workloads.grid_uniform(12, 12, 256, seed=4)
    w.dV = 1.0
    events, _ = _sharded_run(sdm_mod, w, 2, 6, expect_modes=[1, 1])
    assert events > 200


def test_index_base_limits(sdm_mod):
    s = sdm_mod.SDM(1000, 4)
    s.set_index_base(2 ** 32 - 1000)
    for bad in (-1, 2 ** 32 - 999):
        with pytest.raises(sdm_mod.SdmError) as e:
            s.set_index_base(bad)
        assert e.value.code == -1
    s.close()
