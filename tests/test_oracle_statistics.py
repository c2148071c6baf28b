"""Statistical and closed-form pins of the oracle: Golovin moment closed forms (P6),
the one-step mean-field identity tying SDM to Eq. 2 (P7), and exhaustive
enumeration of the outcome distribution on a 3-droplet cell (P8)."""
from fractions import Fraction
import itertools
import math

import numpy as np
from scipy import stats

import oracle
import workloads


def test_golovin_box_moments_follow_closed_forms():
    # For a(v1,v2) = b(v1+v2) the moment equations of Eq. 1 close for any spectrum:
    #   M1 const,  M0(t) = M0(0) exp(-b M1 t / dV),  M2(t) = M2(0) exp(2 b M1 t / dV).
    w = workloads.golovin_box(2 ** 13)
    xi, v, cell = w.xi.copy(), w.v.copy(), w.cell_id.copy()
    m0_0, m1_0, m2_0 = oracle.moments(xi, v)
    rate = w.kparam * m1_0 / w.dV                     # = N0 b vbar of PAPER.md:320 for the discretised state
    assert abs(rate - 1.5e-3) < 2e-5
    checks = {1200: None, 2400: None, 3600: None}
    for step in range(3600):
        xi, v, cell = oracle.remove_zero(xi, v, cell)
        oracle.step(xi, v, cell, 1, w.dt, w.dV, w.kernel, w.kparam, w.seed, step, want_perm=False)
        t = step + 1
        if t in checks:
            checks[t] = oracle.moments(xi, v)
    for t, (m0, m1, m2) in checks.items():
        assert abs(m1 - m1_0) <= 1e-9 * m1_0                                  # water conserved
        assert abs(m0 / m0_0 / math.exp(-rate * t) - 1) < 0.10, (t, m0 / m0_0)  # +-10 % at 2^13
        ratio2 = m2 / m2_0 / math.exp(2 * rate * t)
        assert 1 / 1.5 < ratio2 < 1.5, (t, ratio2)
    # the paper's printed parameters give tau(3600 s) = 1 - exp(-N0 b vbar t) = 0.9955 (Eq. 7)
    assert abs((1 - checks[3600][0] / m0_0) - 0.995484) < 0.002


def test_one_step_mean_field_identity():
    # E[ -delta sum xi ] = (dt/dV) * sum_{a<b} K_ab xi_a xi_b   when every p <= 1
    rng = np.random.default_rng(0)
    n = 7                                           # odd: one droplet is left unpaired each step
    xi0 = rng.integers(50, 200, n).astype(np.int64)
    v0 = rng.uniform(1.0, 3.0, n)
    b, dt, dV = 2.0e-5, 1.0, 1.0
    cell = np.zeros(n, dtype=np.int32)
    expect = 0.0
    for a, c in itertools.combinations(range(n), 2):
        expect += dt / dV * oracle.kernel(0, b, v0[a], v0[c]) * float(xi0[a]) * float(xi0[c])
    pmax = b * 6.0 * 200 * n
    assert pmax < 1.0
    trials = 60000
    dec = np.empty(trials)
    for s in range(trials):
        xi, v = xi0.copy(), v0.copy()
        oracle.step(xi, v, cell, 1, dt, dV, 0, b, 123, s, want_perm=False)
        dec[s] = xi0.sum() - xi.sum()
    se = dec.std(ddof=1) / math.sqrt(trials)
    assert abs(dec.mean() - expect) < 4.5 * se, (dec.mean(), expect, se)
    assert se < 0.05 * expect                        # the test has power


def _enumerate_outcomes(xi, v, b, dt, dV):
    """Exact outcome distribution of one step on a single cell by brute force over all orders
    of the droplets and the position of u relative to frac(p); returns {state: probability}."""
    n = len(xi)
    ratio = Fraction(n * (n - 1) // 2, n // 2)
    out = {}
    perms = list(itertools.permutations(range(n)))
    for order in perms:
        branches = [(Fraction(1, len(perms)), list(xi), list(v))]
        for m in range(n // 2):
            a, c = order[2 * m], order[2 * m + 1]
            nxt = []
            for pr, X, V in branches:
                j, k = (a, c) if X[a] >= X[c] else (c, a)
                p = Fraction(b) * (V[j] + V[k]) * X[j] * ratio * Fraction(dt) / Fraction(dV)
                fl = p.numerator // p.denominator
                frac = p - fl
                for gam, w in ((fl + 1, frac), (fl, 1 - frac)):
                    if w == 0:
                        continue
                    X2, V2 = list(X), list(V)
                    g = min(gam, X2[j] // X2[k])
                    if g > 0:
                        if X2[j] - g * X2[k] > 0:
                            X2[j] -= g * X2[k]
                            V2[k] = V2[k] + g * V2[j]
                        else:
                            V2[j] = V2[k] = V2[k] + g * V2[j]
                            X2[j], X2[k] = X2[k] // 2, X2[k] - X2[k] // 2
                    nxt.append((pr * w, X2, V2))
            branches = nxt
        for pr, X, V in branches:
            key = (tuple(X), tuple(float(x) for x in V))
            out[key] = out.get(key, 0) + pr
    return out


def _check_enumeration(xi, v, b, trials, seed):
    dist = _enumerate_outcomes([int(x) for x in xi], [Fraction(float(x)) for x in v], b, 1.0, 1.0)
    assert sum(dist.values()) == 1
    cell = np.zeros(len(xi), dtype=np.int32)
    seen = {}
    for s in range(trials):
        X, V = xi.copy(), v.copy()
        oracle.step(X, V, cell, 1, 1.0, 1.0, 0, b, seed, s, want_perm=False)
        key = (tuple(int(x) for x in X), tuple(float(x) for x in V))
        seen[key] = seen.get(key, 0) + 1
    assert set(seen) <= set(dist), "oracle produced an outcome the definition does not allow"
    keys = [k for k in dist if dist[k] * trials >= 5]
    obs = np.array([seen.get(k, 0) for k in keys], dtype=float)
    exp = np.array([float(dist[k]) * trials for k in keys])
    rest_o, rest_e = trials - obs.sum(), trials - exp.sum()
    if rest_e >= 5:
        obs, exp = np.append(obs, rest_o), np.append(exp, rest_e)
    chi2 = ((obs - exp) ** 2 / exp).sum()
    assert chi2 < stats.chi2.ppf(1 - 1e-4, len(exp) - 1), (chi2, len(exp))
    return len(dist)


def test_outcome_distribution_three_droplets_bruteforce():
    # n_s = 3 (ratio 3, one droplet unpaired), p spans below and above 1, cap and split reachable
    xi = np.array([3, 2, 1], dtype=np.int64)
    v = np.array([1.0, 2.0, 4.0])
    n_out = _check_enumeration(xi, v, 0.03125, 20000, seed=77)
    assert n_out >= 6


def test_outcome_distribution_two_and_four_droplets_bruteforce():
    _check_enumeration(np.array([4, 2], dtype=np.int64), np.array([1.0, 3.0]), 0.046875, 8000, seed=5)
    _check_enumeration(np.array([2, 2, 1, 3], dtype=np.int64), np.array([1.0, 2.0, 1.0, 0.5]), 0.03125, 30000, seed=6)
