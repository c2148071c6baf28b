"""GPU parity for NEXT-4: cell ids that change between steps (particle displacement happens outside the API,
PAPER.md:223; sdm_set_cell_id), so the cell index (row a2) and the sort by cell carry new work every step."""
import numpy as np
import pytest

import oracle
import workloads

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


def _displace(cell, nx, ny, rng, p_move):
    """Synthetic advection: with probability p_move a droplet hops to a neighbouring cell (periodic grid)."""
    ix, iy = cell % nx, cell // nx
    move = rng.random(cell.shape[0]) < p_move
    dx = rng.integers(-1, 2, cell.shape[0])
    dy = rng.integers(-1, 2, cell.shape[0])
    ix = np.where(move, (ix + dx) % nx, ix)
    iy = np.where(move, (iy + dy) % ny, iy)
    return (iy * nx + ix).astype(np.int32)


@pytest.mark.parametrize("contiguous_start", [True, False])
def test_displacement_between_steps(sdm_mod, contiguous_start):
    nx = ny = 24
    w = workloads.grid_small_multiplicity(nx, ny, 40, shuffled=not contiguous_start, seed=8)
    rng = np.random.default_rng(99)
    s = sdm_mod.SDM(w.n_sd, w.n_cell)
    s.set_state(_dev(w.xi), _dev(w.v), _dev(w.cell_id))
    assert s.counters()["mode"] == (1 if contiguous_start else 0)
    xi, v, cell = w.xi.copy(), w.v.copy(), w.cell_id.copy()
    events = 0
    for step in range(14):
        xi, v, cell = oracle.remove_zero(xi, v, cell)
        assert s.remove_zero() == len(xi)
        if step > 0:                                        # displacement, then the coalescence step (Fig. 3 order)
            cell = _displace(cell, nx, ny, rng, 0.3)
            s.set_cell_id(_dev(cell))
            assert s.counters()["mode"] == 0                # storage is no longer cell-contiguous
        idx, cs, nev = oracle.step(xi, v, cell, w.n_cell, w.dt, w.dV, w.kernel, w.kparam, w.seed, step)
        events += nev
        s.coalescence_step(w.dt, w.dV, w.kernel, w.kparam, w.seed, step)
        gidx, gcs = (t.cpu().numpy() for t in s.get_permutation(len(xi)))
        gxi, gv, gc = (t.cpu().numpy() for t in s.get_state())
        assert np.array_equal(gc, cell) and np.array_equal(gcs, cs) and np.array_equal(gidx, idx), step
        assert np.array_equal(gxi, xi) and np.array_equal(gv, v), step
    assert events > 3000 and len(xi) < w.n_sd
    pm0, pm1, _ = s.moments_host(per_cell=True)
    o0, o1, _ = oracle.moments(xi, v, cell, w.n_cell, per_cell=True)
    assert np.array_equal(pm0, o0) and np.all(np.abs(pm1 - o1) <= 1e-12 * np.maximum(o1, 1e-300))
    s.close()


def test_cells_that_fill_up_switch_to_split_segments_and_back_to_the_fused_path(sdm_mod):
    # everything moves into two cells (700 and 300 droplets: split into key buckets), later back to sorted storage
    rng = np.random.default_rng(5)
    n, n_cell = 1000, 16
    xi = rng.integers(1, 60, n).astype(np.int64)
    v = rng.uniform(0.5, 2.0, n)
    cell = np.sort(rng.integers(0, n_cell, n)).astype(np.int32)
    s = sdm_mod.SDM(n, n_cell)
    s.set_state(_dev(xi), _dev(v), _dev(cell))
    layouts = [np.where(np.arange(n) % 10 < 7, 3, 9).astype(np.int32),
               np.sort(rng.integers(0, n_cell, n)).astype(np.int32)]
    modes = [0, 1]
    step = 0
    for new_cell, mode in zip(layouts, modes):
        s.set_cell_id(_dev(new_cell))
        cnt = s.counters()
        assert cnt["mode"] == mode and cnt["max_cell"] == np.bincount(new_cell, minlength=n_cell).max()
        for _ in range(3):
            idx, cs, _ = oracle.step(xi, v, new_cell, n_cell, 1.0, 1.0, 0, 0.0005, 4, step)
            s.coalescence_step(1.0, 1.0, 0, 0.0005, 4, step)
            gidx, gcs = (t.cpu().numpy() for t in s.get_permutation(n))
            gxi, gv, _ = (t.cpu().numpy() for t in s.get_state())
            assert np.array_equal(gidx, idx) and np.array_equal(gcs, cs)
            assert np.array_equal(gxi, xi) and np.array_equal(gv, v)
            step += 1
    with pytest.raises(sdm_mod.SdmError) as e:
        s.set_cell_id(_dev(np.full(n, n_cell, dtype=np.int32)))
    assert e.value.code == -1
    with pytest.raises(sdm_mod.SdmError) as e:
        s.coalescence_step(1.0, 1.0, 0, 1.0, 0, 0)
    assert e.value.code == -4
    s.close()
