"""GPU parity for NEXT-2: the gravitational kernel with a user-supplied collection-efficiency table
(SDM_KERNEL_GRAVITATIONAL_TABULATED; R16) on every pair path."""
import math

import numpy as np
import pytest

import oracle
import workloads

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

TAB = 2   # KERNEL_GRAVITATIONAL_TABULATED


@pytest.fixture(scope="module")
def sdm_mod():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2101_06318_b200 as m
    m.load_library()
    return m


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _table(n_r=24, seed=0):
    """A Hall-like synthetic table: efficiencies rise with the size of the larger droplet, with noise."""
    rng = np.random.default_rng(seed)
    grid = np.exp(np.linspace(math.log(2e-6), math.log(1.5e-3), n_r))
    big = np.maximum(grid[:, None], grid[None, :])
    E = np.clip((big / 60e-6) ** 1.5, 0.0, 1.0) * rng.uniform(0.5, 1.0, (n_r, n_r))
    E = 0.5 * (E + E.T)
    return grid, E


def _run(sdm_mod, w, steps, grid, E, options=(), expect_mode=None):
    oracle.set_efficiency_table(grid, E)
    s = sdm_mod.SDM(w.n_sd, w.n_cell)
    for k, val in options:
        s.set_option(k, val)
    s.set_efficiency_table(grid, E)
    s.set_state(_dev(w.xi), _dev(w.v), _dev(w.cell_id))
    if expect_mode is not None:
        assert s.counters()["mode"] == expect_mode
    xi, v, cell = w.xi.copy(), w.v.copy(), w.cell_id.copy()
    events = 0
    for step in range(steps):
        xi, v, cell = oracle.remove_zero(xi, v, cell)
        assert s.remove_zero() == len(xi)
        idx, cs, nev = oracle.step(xi, v, cell, w.n_cell, w.dt, w.dV, TAB, w.kparam, w.seed, step)
        events += nev
        s.coalescence_step(w.dt, w.dV, TAB, w.kparam, w.seed, step)
        gidx, _ = (t.cpu().numpy() for t in s.get_permutation(len(xi)))
        gxi, gv, _ = (t.cpu().numpy() for t in s.get_state())
        assert np.array_equal(gidx, idx), f"permutation differs at step {step}"
        assert np.array_equal(gxi, xi), f"multiplicities differ at step {step}"
        assert np.array_equal(gv, v), f"volumes differ at step {step}"
    assert s.counters()["events"] == events
    s.close()
    return events


def test_tabulated_kernel_fused_counting_sort_kernel_with_screening(sdm_mod):
    w = workloads.grid_uniform(16, 16, 256, seed=3)
    w.dV = 0.25
    grid, E = _table()
    assert _run(sdm_mod, w, 6, grid, E, expect_mode=1) > 100


def test_tabulated_kernel_fused_bitonic_kernel_and_screening_off(sdm_mod):
    w = workloads.grid_uniform(24, 24, 64, seed=4)
    w.dV = 0.05
    grid, E = _table(n_r=7, seed=1)
    a = _run(sdm_mod, w, 5, grid, E, expect_mode=1)
    b = _run(sdm_mod, w, 5, grid, E, options=[(sdm_mod.OPT_SCREENING, 0)], expect_mode=1)
    assert a == b > 50


@pytest.mark.parametrize("path", ["box", "general"])
def test_tabulated_kernel_single_cell_box(sdm_mod, path):
    w = workloads.gravitational_box(2 ** 14)
    w.dV = 1e6 / 256
    grid, E = _table(n_r=64, seed=2)
    opts, mode = ([(sdm_mod.OPT_FORCE_GENERAL, 1)], 0) if path == "general" else ([], 2)
    assert _run(sdm_mod, w, 8, grid, E, options=opts, expect_mode=mode) > 50


def test_unit_table_reproduces_the_plain_gravitational_kernel(sdm_mod):
    w = workloads.grid_uniform(8, 8, 256, seed=6)
    w.dV = 0.5
    grid = np.array([1e-6, 1e-3])
    a = sdm_mod.SDM(w.n_sd, w.n_cell)
    b = sdm_mod.SDM(w.n_sd, w.n_cell)
    b.set_efficiency_table(grid, np.ones((2, 2)))
    for s in (a, b):
        s.set_state(_dev(w.xi), _dev(w.v), _dev(w.cell_id))
    for step in range(4):
        a.coalescence_step(w.dt, w.dV, sdm_mod.KERNEL_GRAVITATIONAL, 0.75, 1, step)
        b.coalescence_step(w.dt, w.dV, TAB, 0.75, 1, step)
    for ta, tb in zip(a.get_state(), b.get_state()):
        assert torch.equal(ta, tb)
    assert a.counters()["events"] == b.counters()["events"] > 0
    a.close(), b.close()


def test_efficiency_table_errors(sdm_mod):
    s = sdm_mod.SDM(8, 1)
    s.set_state(_dev(np.ones(4, dtype=np.int64)), _dev(np.ones(4)), _dev(np.zeros(4, dtype=np.int32)))
    with pytest.raises(sdm_mod.SdmError) as e:                 # no table yet
        s.coalescence_step(1.0, 1.0, TAB, 1.0, 0, 0)
    assert e.value.code == -1
    for grid, tab in ((np.array([1.0]), np.ones((1, 1))), (np.array([2.0, 1.0]), np.ones((2, 2))),
                      (np.array([1.0, 2.0]), -np.ones((2, 2))), (np.array([1.0, 2.0]), np.full((2, 2), np.inf)),
                      (np.linspace(1.0, 2.0, 65), np.ones((65, 65)))):
        with pytest.raises(sdm_mod.SdmError) as e:
            s.set_efficiency_table(grid, tab)
        assert e.value.code == -1
    s.set_efficiency_table(np.array([1.0, 2.0]), np.ones((2, 2)))
    s.coalescence_step(1.0, 1.0, TAB, 1.0, 0, 0)
    s.close()
