"""GPU parity at BASELINE.json's FULL sizes and FULL lengths, driven through the same
C-ABI calls bench.py uses:

    C1  Golovin box 2^13           3600 steps, state vs oracle every 300
    C2  Golovin box 2^17           3600 steps, state + permutation vs oracle every 100; closed forms
        Golovin box 2^20           300 steps vs oracle every 50, then the GPU alone to 3600 s; closed forms
    C3  gravitational box 2^14     3600 steps at the config's own dV, every 300
        gravitational box 2^20     100 steps, every 25
    C4  128x128 Poisson(64) grid   600 steps with removal every step, both storage layouts, every 50
    C5  512x512x256 = 2^26         real parameters (dV = 1e3): 3 steps with the WHOLE state and WHOLE idx
                                   against oracle.step on the full arrays, then 12 steps in total checked on
                                   every cell that changed plus 256 random cells (per-cell oracle)

The state after k steps pins every earlier step (one wrong pair changes xi for good).  The oracle
trajectories run concurrently in a small thread pool (tests/conftest.py: the oracle itself is unchanged,
one thread per trajectory) so that the whole file fits the GPU-test time budget."""
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


# name -> (workload factory, checkpoints [steps]); submitted longest first
JOBS = {
    "C4s": (lambda: workloads.grid_poisson(shuffled=True), range(50, 601, 50)),
    "C4c": (lambda: workloads.grid_poisson(shuffled=False), range(50, 601, 50)),
    "C2a": (lambda: workloads.golovin_box(2 ** 17), range(100, 3601, 100)),
    "C2b": (lambda: workloads.golovin_box(2 ** 20), range(50, 301, 50)),
    "C3b": (lambda: workloads.gravitational_box(2 ** 20), range(25, 101, 25)),
    "C3a": (lambda: workloads.gravitational_box(2 ** 14), range(300, 3601, 300)),
    "C1": (lambda: workloads.golovin_box(2 ** 13), range(300, 3601, 300)),
}


@pytest.fixture(scope="module")
def trajectories(sdm_mod, oracle_pool):
    """All oracle trajectories of this file, started together at first use."""
    return {name: oracle_pool(name, make, cps) for name, (make, cps) in JOBS.items()}


def _load(sdm_mod, w):
    s = sdm_mod.SDM(w.n_sd, w.n_cell)
    s.set_state_host(torch.from_numpy(w.xi).pin_memory(), torch.from_numpy(w.v).pin_memory(),
                     torch.from_numpy(w.cell_id).pin_memory())
    return s


def _assert_state_equal(s, xi, v, cell, what):
    gxi, gv, gc = (t.cpu().numpy() for t in s.get_state())
    assert len(gxi) == len(xi), f"{what}: survivor count {len(gxi)} != {len(xi)}"
    assert np.array_equal(gc, cell), f"{what}: cell ids differ"
    assert np.array_equal(gxi, xi), f"{what}: multiplicities differ"
    assert np.array_equal(gv, v), f"{what}: volumes differ, max rel {np.max(np.abs(gv - v) / v):.3e} (bar 1e-12)"


def _follow(s, traj, what, per_step_calls_at=()):
    """Drives the GPU through the trajectory's checkpoints with sdm_run ([remove_zero; step] per step) and
    compares state, permutation and cell table of the last step, and the event counter at every one of them.
    Checkpoints listed in per_step_calls_at are reached through the per-step entry points instead."""
    w = traj.w
    snaps = traj.result()
    t = 0
    for cp, (xi, v, cell, idx, cs, events) in zip(traj.checkpoints, snaps):
        if cp in per_step_calls_at:
            for step in range(t, cp):
                s.remove_zero(sync=False)
                s.coalescence_step(w.dt, w.dV, w.kernel, w.kparam, w.seed, step)
        else:
            s.run(w.dt, w.dV, w.kernel, w.kparam, w.seed, t, cp - t, True)
        t = cp
        _assert_state_equal(s, xi, v, cell, f"{what} after {cp} steps")
        gidx, gcs = (a.cpu().numpy() for a in s.get_permutation(len(xi)))
        assert np.array_equal(gcs, cs), f"{what}: cell_start of step {cp - 1} differs"
        assert np.array_equal(gidx, idx), f"{what}: permutation of step {cp - 1} differs"
        assert s.counters()["events"] == events, f"{what}: event count after {cp} steps"
    return snaps[-1]


def _golovin_check(w, m_init, m_now, t, tol_m0):
    """Closed forms for a = b (v1 + v2), any initial spectrum: M1 const, M0(t) = M0(0) exp(-b M1 t / dV),
    M2(t) = M2(0) exp(2 b M1 t / dV)  (moment equations of Eq. 1; tau of Eq. 7)."""
    rate = w.kparam * m_init[1] / w.dV
    assert abs(m_now[1] - m_init[1]) <= 1e-9 * m_init[1], "water not conserved"
    r0 = m_now[0] / m_init[0] / math.exp(-rate * t)
    assert abs(r0 - 1) < tol_m0, (t, r0)
    r2 = m_now[2] / m_init[2] / math.exp(2 * rate * t)
    assert 1 / 1.5 < r2 < 1.5, (t, r2)


def _moments_match(s, xi, v):
    m = s.moments_host()
    o = oracle.moments(xi, v)
    assert m[0] == o[0] and abs(m[1] - o[1]) <= 1e-12 * o[1] and abs(m[2] - o[2]) <= 1e-12 * o[2]
    return m


def test_c5_real_parameters_whole_state_three_steps_then_changed_cells(sdm_mod, trajectories):
    """Config 5 as bench.py times it (dV = 1e3, xi = 1e6, gravitational, 2^26 droplets, remove_zero +
    step_moments).  Steps 0-2: oracle.step on the FULL arrays, everything compared (xi, v, idx, cell_start,
    moments).  Steps 3-11 on the GPU alone; then every cell whose state changed in the 12 steps plus 256
    random cells is recomputed by the oracle from the initial state (cells are independent and the Philox
    counter is the global storage index): state and the permutation of the last step."""
    w = workloads.grid_uniform(512, 512, 256, seed=0)
    assert w.dV == 1e3 and w.n_sd == 2 ** 26
    s = _load(sdm_mod, w)
    assert s.counters()["mode"] == 1
    mom = s.moments()
    xi, v = w.xi.copy(), w.v.copy()
    events = 0
    for step in range(3):
        s.remove_zero(sync=False)
        s.coalescence_step_moments(w.dt, w.dV, w.kernel, w.kparam, w.seed, step, out=mom)
        idx, cs, nev = oracle.step(xi, v, w.cell_id, w.n_cell, w.dt, w.dV, w.kernel, w.kparam, w.seed, step)
        events += nev
        gidx, gcs = s.get_permutation(w.n_sd)
        assert np.array_equal(gcs.cpu().numpy(), cs), f"cell_start of step {step}"
        assert np.array_equal(gidx.cpu().numpy(), idx), f"whole permutation of step {step}"
        del gidx, idx
        gxi, gv, gc = s.get_state()
        assert np.array_equal(gxi.cpu().numpy(), xi), f"whole xi after step {step}"
        assert np.array_equal(gv.cpu().numpy(), v), f"whole v after step {step}"
        assert np.array_equal(gc.cpu().numpy(), w.cell_id)
        del gxi, gv, gc
        o0, o1, o2 = oracle.moments(xi, v)
        assert int(mom[0].cpu()[0]) == o0
        assert abs(float(mom[1].cpu()[0]) - o1) <= 1e-12 * o1 and abs(float(mom[2].cpu()[0]) - o2) <= 1e-12 * o2
    assert events > 500 and s.counters()["events"] == events
    n_steps = 12
    for step in range(3, n_steps):
        s.remove_zero(sync=False)
        s.coalescence_step_moments(w.dt, w.dV, w.kernel, w.kparam, w.seed, step, out=mom)
    gxi, gv, _ = s.get_state()
    hxi, hv = gxi.cpu().numpy(), gv.cpu().numpy()
    hidx = s.get_permutation(w.n_sd)[0].cpu().numpy()
    del gxi, gv
    assert len(hxi) == w.n_sd
    changed = np.unique(np.nonzero((hxi != w.xi) | (hv != w.v))[0] // 256)
    assert len(changed) > 2000
    rng = np.random.default_rng(123)
    sample = np.unique(np.concatenate([changed, rng.integers(0, w.n_cell, 256), [0, w.n_cell - 1]]))
    zc = np.zeros(256, dtype=np.int32)
    total_events = 0
    for c in sample:
        lo, hi = int(c) * 256, int(c) * 256 + 256
        xs, vs = w.xi[lo:hi].copy(), w.v[lo:hi].copy()
        sid = np.arange(lo, hi, dtype=np.int64)
        for step in range(n_steps):
            li, _, nev = oracle.step(xs, vs, zc, 1, w.dt, w.dV, w.kernel, w.kparam, w.seed, step, sid=sid,
                                     want_perm=(step == n_steps - 1))
            total_events += nev
        assert np.array_equal(lo + li, hidx[lo:hi]), f"permutation of cell {c}"
        assert np.array_equal(xs, hxi[lo:hi]) and np.array_equal(vs, hv[lo:hi]), f"state of cell {c}"
    assert total_events == s.counters()["events"]          # every event of the run lies in a compared cell
    assert int(mom[0].cpu()[0]) == int(hxi.sum())
    s.close()


def test_c1_golovin_box_2e13_all_3600_steps_and_closed_forms(sdm_mod, trajectories):
    traj = trajectories["C1"]
    w = traj.w
    s = _load(sdm_mod, w)
    assert s.counters()["mode"] == 2                          # single-cell box: the persistent box path
    m_init = s.moments_host()
    assert m_init[0] == 2 ** 23 * 10 ** 6
    xi, v, cell, _, _, events = _follow(s, traj, "C1", per_step_calls_at=(300,))
    _golovin_check(w, m_init, _moments_match(s, xi, v), 3600, 0.10)
    assert events > 30000 and s.counters()["n_sd"] == len(xi)
    s.close()


def test_c2_golovin_box_2e17_all_3600_steps_and_closed_forms(sdm_mod, trajectories):
    """Config 2 at n = 2^17 in full: 3600 steps, everything compared with the oracle every 100 steps; moments
    against the Golovin closed forms at t = 1200, 2400, 3600 s."""
    traj = trajectories["C2a"]
    w = traj.w
    s = _load(sdm_mod, w)
    m_init = s.moments_host()
    snaps = traj.result()
    xi, v, cell, _, _, events = _follow(s, traj, "C2 2^17")
    for cp, snap in zip(traj.checkpoints, snaps):
        if cp % 1200 == 0:
            o = oracle.moments(snap[0], snap[1])
            _golovin_check(w, m_init, o, cp, 0.05)
    m = _moments_match(s, xi, v)
    _golovin_check(w, m_init, m, 3600, 0.05)
    assert abs((1 - m[0] / m_init[0]) - 0.995484) < 0.003    # tau(3600 s) of Eq. 7 with the paper's parameters
    assert events > 100000
    s.close()


def test_c2_golovin_box_2e20_300_steps_then_closed_forms(sdm_mod, trajectories):
    """Config 2 at n = 2^20: 300 steps against the oracle (every 50), then the GPU alone to t = 3600 s with
    moments against the Golovin closed forms at t = 1200, 2400, 3600 s."""
    traj = trajectories["C2b"]
    w = traj.w
    s = _load(sdm_mod, w)
    m_init = s.moments_host()
    xi, v, cell, _, _, events = _follow(s, traj, "C2 2^20")
    assert events > 10000
    t, m_prev = 300, _moments_match(s, xi, v)
    for t_out in (1200, 2400, 3600):
        s.run(w.dt, w.dV, w.kernel, w.kparam, w.seed, t, t_out - t, True)
        t = t_out
        m = s.moments_host()
        assert m[0] <= m_prev[0]
        _golovin_check(w, m_init, m, t, 0.05)
        m_prev = m
    assert abs((1 - m_prev[0] / m_init[0]) - 0.995484) < 0.002
    s.close()


def test_c3_gravitational_box_2e14_all_3600_steps(sdm_mod, trajectories):
    """Config 3's kernel and dV at n = 2^14 ("parity 3600 steps at n = 2^14")."""
    traj = trajectories["C3a"]
    s = _load(sdm_mod, traj.w)
    m1_0 = s.moments_host()[1]
    xi, v, cell, _, _, events = _follow(s, traj, "C3 2^14")
    m = _moments_match(s, xi, v)
    assert abs(m[1] - m1_0) <= 1e-9 * m1_0 and events > 1000
    s.close()


def test_c3_gravitational_box_2e20_100_steps(sdm_mod, trajectories):
    """Config 3 at its full size with the paper's dV: 100 steps against the oracle, every 25."""
    traj = trajectories["C3b"]
    s = _load(sdm_mod, traj.w)
    assert s.counters()["mode"] == 2
    m1_0 = s.moments_host()[1]
    xi, v, cell, _, _, events = _follow(s, traj, "C3 2^20", per_step_calls_at=(25,))
    m = _moments_match(s, xi, v)
    assert abs(m[1] - m1_0) <= 1e-9 * m1_0 and m[0] < 2 ** 23 * 10 ** 6 and events > 1000
    s.close()


@pytest.mark.parametrize("shuffled", [True, False])
def test_c4_poisson_grid_128x128_all_600_steps(sdm_mod, trajectories, shuffled):
    """Config 4 at its full size (1 048 760 droplets in 16 384 cells of 31..98) with the paper's parameters,
    zero removal every step, both storage layouts: all 600 steps, compared every 50."""
    traj = trajectories["C4s" if shuffled else "C4c"]
    w = traj.w
    assert w.n_sd == 1048760 and w.notes["count_min"] == 31 and w.notes["count_max"] == 98
    s = _load(sdm_mod, w)
    assert s.counters()["mode"] == (0 if shuffled else 1)
    xi, v, cell, _, _, events = _follow(s, traj, "C4 shuffled" if shuffled else "C4 contiguous",
                                        per_step_calls_at=(50,))
    pm0, pm1, pm2 = s.moments_host(per_cell=True)
    o0, o1, o2 = oracle.moments(xi, v, cell, w.n_cell, per_cell=True)
    assert np.array_equal(pm0, o0) and np.all(np.abs(pm1 - o1) <= 1e-12 * o1) and np.all(np.abs(pm2 - o2) <= 1e-12 * o2)
    assert events > 0
    s.close()
