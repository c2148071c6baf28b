"""GPU parity at BASELINE.json's FULL sizes (configs 1-4; config 5 is in test_gpu_parity.py), driven
through the same C-ABI calls bench.py uses, plus the Golovin closed forms of the moments (PAPER.md:
305-320) on the GPU's own 3600-step runs.

Sizes the oracle cannot run for the full number of steps within a test budget are compared on a
prefix of the steps (the state after k steps pins every earlier step: one wrong pair changes xi for
good), and the rest of the run is checked through what holds at any size: conservation of water,
monotone non-increasing total multiplicity, and the closed forms."""
import math

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


def _load(sdm_mod, w):
    s = sdm_mod.SDM(w.n_sd, w.n_cell)
    s.set_state_host(torch.from_numpy(w.xi).pin_memory(), torch.from_numpy(w.v).pin_memory(),
                     torch.from_numpy(w.cell_id).pin_memory())
    return s


def _oracle_advance(w, xi, v, cell, step0, n_steps):
    events = 0
    for step in range(step0, step0 + n_steps):
        xi, v, cell = oracle.remove_zero(xi, v, cell)
        _, _, nev = oracle.step(xi, v, cell, w.n_cell, w.dt, w.dV, w.kernel, w.kparam, w.seed, step,
                                want_perm=False)
        events += nev
    return xi, v, cell, events


def _assert_state_equal(s, xi, v, cell, what):
    gxi, gv, gc = (t.cpu().numpy() for t in s.get_state())
    assert len(gxi) == len(xi), f"{what}: survivor count {len(gxi)} != {len(xi)}"
    assert np.array_equal(gc, cell), f"{what}: cell ids differ"
    assert np.array_equal(gxi, xi), f"{what}: multiplicities differ"
    assert np.array_equal(gv, v), f"{what}: volumes differ, max rel {np.max(np.abs(gv - v) / v):.3e} (bar 1e-12)"


def _check_permutation_of_last_step(s, w, xi_before, v_before, cell_before, step):
    """idx / cell_start of the GPU's last step against the oracle's for the same pre-step state."""
    xi, v = xi_before.copy(), v_before.copy()
    idx, cs, nev = oracle.step(xi, v, cell_before, w.n_cell, w.dt, w.dV, w.kernel, w.kparam, w.seed, step)
    gidx, gcs = (t.cpu().numpy() for t in s.get_permutation(len(xi)))
    assert np.array_equal(gcs, cs) and np.array_equal(gidx, idx), f"permutation of step {step} differs"
    return xi, v, nev


def _golovin_check(w, m_init, m_now, t, tol_m0):
    """Closed forms for a = b (v1 + v2), any initial spectrum: M1 const, M0(t) = M0(0) exp(-b M1 t / dV),
    M2(t) = M2(0) exp(2 b M1 t / dV)  (moment equations of Eq. 1; tau of Eq. 7)."""
    rate = w.kparam * m_init[1] / w.dV
    assert abs(m_now[1] - m_init[1]) <= 1e-9 * m_init[1], "water not conserved"
    r0 = m_now[0] / m_init[0] / math.exp(-rate * t)
    assert abs(r0 - 1) < tol_m0, (t, r0)
    r2 = m_now[2] / m_init[2] / math.exp(2 * rate * t)
    assert 1 / 1.5 < r2 < 1.5, (t, r2)


def test_c1_golovin_box_2e13_all_3600_steps_and_closed_forms(sdm_mod):
    """Config 1 in full: 3600 steps, state compared with the oracle every 300 steps and at the end."""
    w = workloads.golovin_box(2 ** 13)
    s = _load(sdm_mod, w)
    assert s.counters()["mode"] == 0
    m_init = s.moments_host()
    assert m_init[0] == 2 ** 23 * 10 ** 6
    xi, v, cell = w.xi.copy(), w.v.copy(), w.cell_id.copy()
    events = 0
    for t0 in range(0, 3600, 300):
        s.run(w.dt, w.dV, w.kernel, w.kparam, w.seed, t0, 300, True)
        xi, v, cell, nev = _oracle_advance(w, xi, v, cell, t0, 300)
        events += nev
        _assert_state_equal(s, xi, v, cell, f"C1 after {t0 + 300} steps")
        if (t0 + 300) % 1200 == 0:
            m = s.moments_host()
            o = oracle.moments(xi, v)
            assert m[0] == o[0] and abs(m[1] - o[1]) <= 1e-12 * o[1] and abs(m[2] - o[2]) <= 1e-12 * o[2]
            _golovin_check(w, m_init, m, t0 + 300, 0.10)
    cnt = s.counters()
    assert cnt["events"] == events > 30000 and cnt["n_sd"] == len(xi)
    s.close()


@pytest.mark.parametrize("log2n,parity_steps,tol", [(17, 240, 0.05), (20, 12, 0.05)])
def test_c2_golovin_box_full_size_prefix_parity_then_closed_forms(sdm_mod, log2n, parity_steps, tol):
    """Config 2 at n = 2^17 and 2^20: bit-exact state against the oracle over the first steps
    (permutation checked on the first and the last of them), then the GPU alone to t = 3600 s with
    moments against the Golovin closed forms at t = 1200, 2400, 3600 s."""
    w = workloads.golovin_box(2 ** log2n)
    s = _load(sdm_mod, w)
    m_init = s.moments_host()
    xi, v, cell = w.xi.copy(), w.v.copy(), w.cell_id.copy()
    # step 0 with the permutation
    s.remove_zero(sync=False)
    s.coalescence_step(w.dt, w.dV, w.kernel, w.kparam, w.seed, 0)
    xi, v, _ = _check_permutation_of_last_step(s, w, xi, v, cell, 0)
    _assert_state_equal(s, xi, v, cell, "C2 step 0")
    # steps 1 .. parity_steps-2 through sdm_run
    s.run(w.dt, w.dV, w.kernel, w.kparam, w.seed, 1, parity_steps - 2, True)
    xi, v, cell, events = _oracle_advance(w, xi, v, cell, 1, parity_steps - 2)
    _assert_state_equal(s, xi, v, cell, f"C2 after {parity_steps - 1} steps")
    assert events > 0
    # last parity step, permutation again (the state now holds unequal multiplicities)
    last = parity_steps - 1
    xi, v, cell = oracle.remove_zero(xi, v, cell)
    assert s.remove_zero() == len(xi)
    s.coalescence_step(w.dt, w.dV, w.kernel, w.kparam, w.seed, last)
    xi, v, _ = _check_permutation_of_last_step(s, w, xi, v, cell, last)
    _assert_state_equal(s, xi, v, cell, f"C2 step {last}")
    # the rest of the hour on the GPU alone
    t, m_prev = parity_steps, s.moments_host()
    for t_out in (1200, 2400, 3600):
        s.run(w.dt, w.dV, w.kernel, w.kparam, w.seed, t, t_out - t, True)
        t = t_out
        m = s.moments_host()
        assert m[0] <= m_prev[0]
        _golovin_check(w, m_init, m, t, tol)
        m_prev = m
    # tau(3600 s) of Eq. 7 with the paper's printed parameters: 1 - exp(-N0 b vbar t) = 0.995484
    assert abs((1 - m_prev[0] / m_init[0]) - 0.995484) < 0.002
    cnt = s.counters()
    assert cnt["zeros"] >= 0 and cnt["n_sd"] <= w.n_sd
    s.close()


def test_c3_gravitational_box_2e20_parity(sdm_mod):
    """Config 3 at its full size, gravitational kernel with the paper's dV: 10 steps against the oracle."""
    w = workloads.gravitational_box(2 ** 20)
    s = _load(sdm_mod, w)
    assert s.counters()["mode"] == 0
    xi, v, cell = w.xi.copy(), w.v.copy(), w.cell_id.copy()
    m1_0 = oracle.moments(xi, v)[1]
    s.run(w.dt, w.dV, w.kernel, w.kparam, w.seed, 0, 9, True)
    xi, v, cell, events = _oracle_advance(w, xi, v, cell, 0, 9)
    _assert_state_equal(s, xi, v, cell, "C3 after 9 steps")
    xi, v, cell = oracle.remove_zero(xi, v, cell)
    assert s.remove_zero() == len(xi)
    s.coalescence_step(w.dt, w.dV, w.kernel, w.kparam, w.seed, 9)
    xi, v, _ = _check_permutation_of_last_step(s, w, xi, v, cell, 9)
    _assert_state_equal(s, xi, v, cell, "C3 step 9")
    m = s.moments_host()
    assert abs(m[1] - m1_0) <= 1e-12 * m1_0 and m[0] < 2 ** 23 * 10 ** 6
    assert events > 100
    s.close()


@pytest.mark.parametrize("shuffled", [True, False])
def test_c4_poisson_grid_128x128_full_size(sdm_mod, shuffled):
    """Config 4 at its full size (1 048 760 droplets in 16 384 cells of 31..98), zero removal every
    step, both storage layouts: 20 steps against the oracle with the paper's parameters."""
    w = workloads.grid_poisson(shuffled=shuffled)
    assert w.n_sd == 1048760 and w.notes["count_min"] == 31 and w.notes["count_max"] == 98
    s = _load(sdm_mod, w)
    assert s.counters()["mode"] == (0 if shuffled else 1)
    xi, v, cell = w.xi.copy(), w.v.copy(), w.cell_id.copy()
    s.run(w.dt, w.dV, w.kernel, w.kparam, w.seed, 0, 19, True)
    xi, v, cell, events = _oracle_advance(w, xi, v, cell, 0, 19)
    _assert_state_equal(s, xi, v, cell, "C4 after 19 steps")
    xi, v, cell = oracle.remove_zero(xi, v, cell)
    assert s.remove_zero() == len(xi)
    s.coalescence_step(w.dt, w.dV, w.kernel, w.kparam, w.seed, 19)
    xi, v, nev = _check_permutation_of_last_step(s, w, xi, v, cell, 19)
    events += nev
    _assert_state_equal(s, xi, v, cell, "C4 step 19")
    pm0, pm1, pm2 = s.moments_host(per_cell=True)
    o0, o1, o2 = oracle.moments(xi, v, cell, w.n_cell, per_cell=True)
    assert np.array_equal(pm0, o0) and np.all(np.abs(pm1 - o1) <= 1e-12 * o1) and np.all(np.abs(pm2 - o2) <= 1e-12 * o2)
    assert s.counters()["events"] == events
    s.close()
