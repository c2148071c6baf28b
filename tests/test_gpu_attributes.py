"""GPU parity for N_ATTR > 1 extensive attributes:
every attribute row is updated by each coalescence event like the volume, moves with its droplet in
sdm_remove_zero, and never changes the permutation or the multiplicities."""
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


def _attr_block(w, n_attr, seed):
    rng = np.random.default_rng(seed)
    attr = np.empty((n_attr, w.n_sd))
    attr[0] = w.v
    for r in range(1, n_attr):
        attr[r] = rng.uniform(-3.0, 7.0, w.n_sd) if r % 2 else rng.integers(0, 9, w.n_sd).astype(np.float64)
    return attr


def _run(sdm_mod, w, n_attr, steps, options=(), expect_mode=None, seed=21):
    attr = _attr_block(w, n_attr, seed)
    s = sdm_mod.SDM(w.n_sd, w.n_cell, n_attr=n_attr)
    for k, val in options:
        s.set_option(k, val)
    s.set_state(_dev(w.xi), _dev(w.v), _dev(w.cell_id))
    assert torch.count_nonzero(s.get_attributes()) == 0          # zero-filled until sdm_set_attributes
    s.set_attributes(_dev(attr[1:]))
    if expect_mode is not None:
        assert s.counters()["mode"] == expect_mode
    xi, cell = w.xi.copy(), w.cell_id.copy()
    events = 0
    for step in range(steps):
        xi, attr, cell = oracle.remove_zero_attr(xi, attr, cell)
        assert s.remove_zero() == len(xi)
        idx, cs, nev = oracle.step_attr(xi, attr, cell, w.n_cell, w.dt, w.dV, w.kernel, w.kparam, w.seed, step)
        events += nev
        if step % 2:
            s.coalescence_step_moments(w.dt, w.dV, w.kernel, w.kparam, w.seed, step)
        else:
            s.coalescence_step(w.dt, w.dV, w.kernel, w.kparam, w.seed, step)
        gidx, gcs = (t.cpu().numpy() for t in s.get_permutation(len(xi)))
        gxi, gv, gc = (t.cpu().numpy() for t in s.get_state())
        ga = s.get_attributes().cpu().numpy()
        assert np.array_equal(gidx, idx) and np.array_equal(gcs, cs), f"permutation differs at step {step}"
        assert np.array_equal(gxi, xi) and np.array_equal(gc, cell), f"multiplicities differ at step {step}"
        assert np.array_equal(gv, attr[0]), f"volumes differ at step {step}"
        assert np.array_equal(ga, attr[1:]), f"attributes differ at step {step}"
    assert s.counters()["events"] == events
    s.close()
    return events, len(xi)


def test_attributes_fused_path_with_removal(sdm_mod):
    w = workloads.grid_small_multiplicity(24, 24, 32, shuffled=False, seed=3)
    events, n_end = _run(sdm_mod, w, 4, 16, expect_mode=1)
    assert events > 3000 and n_end < w.n_sd


def test_attributes_general_path_with_removal(sdm_mod):
    w = workloads.grid_small_multiplicity(24, 24, 32, shuffled=True, seed=4)
    events, n_end = _run(sdm_mod, w, 3, 16, expect_mode=0)
    assert events > 3000 and n_end < w.n_sd


@pytest.mark.parametrize("path", ["box", "general"])
def test_attributes_single_cell_box_and_max_rows(sdm_mod, path):
    w = workloads.golovin_box(2 ** 12)
    w.kparam = 1500.0 * 200                                   # events from the first step on
    opts, mode = ([(sdm_mod.OPT_FORCE_GENERAL, 1)], 0) if path == "general" else ([], 2)
    events, _ = _run(sdm_mod, w, sdm_mod.binding.MAX_ATTR, 12, options=opts, expect_mode=mode)
    assert events > 500


def test_attributes_gravitational_256_cells_counting_sort_kernel(sdm_mod):
    w = workloads.grid_uniform(12, 12, 256, seed=5)
    w.dV = 1.0
    events, _ = _run(sdm_mod, w, 2, 6, expect_mode=1)
    assert events > 100


def test_compaction_moves_every_row_over_many_tiles(sdm_mod):
    rng = np.random.default_rng(7)
    n = 2048 * 9 + 77
    xi = rng.integers(0, 3, n).astype(np.int64)
    xi[3000:7000] = 0
    v = rng.random(n) + 0.1
    cell = np.sort(rng.integers(0, 40, n)).astype(np.int32)
    extra = rng.standard_normal((7, n))
    s = sdm_mod.SDM(n, 40, n_attr=8)
    s.set_state(_dev(xi), _dev(v), _dev(cell))
    s.set_attributes(_dev(extra))
    keep = xi != 0
    assert s.remove_zero() == int(keep.sum())
    gxi, gv, gc = (t.cpu().numpy() for t in s.get_state())
    assert np.array_equal(gxi, xi[keep]) and np.array_equal(gv, v[keep]) and np.array_equal(gc, cell[keep])
    assert np.array_equal(s.get_attributes().cpu().numpy(), extra[:, keep])
    s.close()


def test_attribute_errors(sdm_mod):
    s = sdm_mod.SDM(8, 1)
    s.set_state(_dev(np.ones(4, dtype=np.int64)), _dev(np.ones(4)), _dev(np.zeros(4, dtype=np.int32)))
    with pytest.raises(sdm_mod.SdmError) as e:
        s._check(s._lib.sdm_set_attributes(s._h, None, 4))
    assert e.value.code == -1                                 # n_attr == 1
    s.close()
    s = sdm_mod.SDM(8, 1, n_attr=2)
    s.set_state(_dev(np.ones(4, dtype=np.int64)), _dev(np.ones(4)), _dev(np.zeros(4, dtype=np.int32)))
    bad = np.ones((1, 4))
    bad[0, 2] = np.nan
    with pytest.raises(sdm_mod.SdmError) as e:
        s.set_attributes(_dev(bad))
    assert e.value.code == -1
    with pytest.raises(sdm_mod.SdmError) as e:
        s.coalescence_step(1.0, 1.0, 0, 1.0, 0, 0)
    assert e.value.code == -4
    s.close()
    with pytest.raises(sdm_mod.SdmError):
        sdm_mod.SDM(8, 1, n_attr=9)
