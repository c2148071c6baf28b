"""Pins for rows a5/a6 of the oracle: Eq. 3, gamma, Eq. 4 cap, Eqs. 5-6 / Fig. 5.
PAPER.md:85, 102-126, 252-287."""
from fractions import Fraction
import math

import numpy as np

import oracle
from conftest import read_golden


def test_paper_fig1b_worked_example():
    g = read_golden("paper_worked_examples.txt")
    xj, xk, gam = int(g["fig1b_xi_j"]), int(g["fig1b_xi_k"]), int(g["fig1b_gamma"])
    # p = 4.5 with u = 0.25 gives gamma = ceil(4.5 - 0.25) = 5
    assert oracle.gamma_tilde(4.5, 0.25, xj, xk) == int(g["fig1b_gamma_tilde"])
    A_j, A_k = 3.0, 7.0
    xa, va, xb, vb = oracle.collide_pair(xj, A_j, xk, A_k, gam)
    assert (xa, xb) == (int(g["fig1b_xi_j_after"]), int(g["fig1b_xi_k_after"]))
    assert va == A_j and vb == A_k + 4 * A_j          # Eq. 5
    # the same pair stored in the other order gives the mirrored result
    xa, va, xb, vb = oracle.collide_pair(xk, A_k, xj, A_j, gam)
    assert (xa, va, xb, vb) == (2, A_k + 4 * A_j, 1, A_j)


def test_paper_xi_k_equal_one_removes_j():
    g = read_golden("paper_worked_examples.txt")
    xa, va, xb, vb = oracle.collide_pair(1, 2.0, 1, 5.0, 1)
    assert (xa, xb) == (int(g["eq6_xi1_xi_j_after"]), int(g["eq6_xi1_xi_k_after"]))
    assert va == vb == 1 * 2.0 + 5.0                   # Eq. 6: both carry g*A_j + A_k


def test_eq6_split_rule_and_tie_orientation():
    # equal multiplicities: strict '<' keeps the first-in-pair as j; j gets floor, k gets the rest
    xa, va, xb, vb = oracle.collide_pair(7, 1.5, 7, 2.5, 3)
    assert (xa, xb) == (3, 4) and va == vb == 1.5 + 2.5
    # xi_j = 3 xi_k exactly with gamma >= 3 -> new_n == 0 -> split of xi_k, attributes g*A_j + A_k
    xa, va, xb, vb = oracle.collide_pair(4, 10.0, 12, 1.0, 99)
    assert (xa, xb) == (2, 2) and va == vb == 3 * 1.0 + 10.0
    # zero gamma: nothing changes; zero-xi partner: nothing changes
    assert oracle.collide_pair(5, 1.0, 3, 2.0, 0) == (5, 1.0, 3, 2.0)
    assert oracle.collide_pair(5, 1.0, 0, 2.0, 4) == (5, 1.0, 0, 2.0)


def test_collide_matches_eq5_eq6_exact_rationals():
    rng = np.random.default_rng(1)
    for _ in range(3000):
        xa, xb = int(rng.integers(1, 40)), int(rng.integers(1, 40))
        va, vb = float(rng.integers(1, 1000)), float(rng.integers(1, 1000))   # exact in fp64
        gam = int(rng.integers(0, 8))
        got = oracle.collide_pair(xa, va, xb, vb, gam)
        # Eqs. 4-6 with j = larger multiplicity (first on ties)
        first_is_j = xa >= xb
        (nj, aj, nk, ak) = (xa, va, xb, vb) if first_is_j else (xb, vb, xa, va)
        gt = min(gam, nj // nk)
        if gt > 0:
            if nj - gt * nk > 0:
                nj, ak = nj - gt * nk, ak + gt * aj
            else:
                aj = ak = ak + gt * aj
                nj, nk = nk // 2, nk - nk // 2
        want = (nj, aj, nk, ak) if first_is_j else (nk, ak, nj, aj)
        assert got == want
        # water conservation for the pair, exactly
        assert Fraction(got[0]) * Fraction(got[1]) + Fraction(got[2]) * Fraction(got[3]) == \
            Fraction(xa) * Fraction(va) + Fraction(xb) * Fraction(vb)


def test_gamma_is_ceil_p_minus_phi_in_exact_arithmetic():
    # PAPER.md:102 gamma = ceil(p - phi); the oracle's floor form must agree with exact rationals
    rng = np.random.default_rng(2)
    big = 10 ** 12
    for _ in range(20000):
        p = float(rng.uniform(0, 6)) if rng.random() < 0.8 else float(rng.integers(0, 6))
        u = float(rng.integers(0, 2 ** 53)) / 2.0 ** 53
        want = math.ceil(Fraction(p) - Fraction(u))
        assert oracle.gamma_tilde(p, u, big, 1) == want
    assert oracle.gamma_tilde(0.0, 0.0, big, 1) == 0
    assert oracle.gamma_tilde(1.0, 0.0, big, 1) == 1
    assert oracle.gamma_tilde(0.3, 0.3, big, 1) == 0       # phi == p: ceil(0) = 0
    assert oracle.gamma_tilde(0.3, np.nextafter(0.3, 0), big, 1) == 1


def test_gamma_cap_and_huge_p():
    assert oracle.gamma_tilde(75.0, 0.5, 5, 2) == 2
    assert oracle.gamma_tilde(1e300, 0.5, 9, 2) == 4            # no overflow in the conversion
    assert oracle.gamma_tilde(float(2 ** 63), 0.5, 2 ** 62, 1) == 2 ** 62
    assert oracle.gamma_tilde(2.5, 0.9, 3, 3) == 1


def test_eq3_probability_against_exact_rational_formula():
    rng = np.random.default_rng(3)
    for _ in range(2000):
        K = float(rng.uniform(1e-12, 1e-6))
        xi = int(rng.integers(1, 10 ** 9))
        n = int(rng.integers(2, 400))
        dt, dV = float(rng.uniform(0.1, 10)), float(rng.uniform(1, 1e6))
        p = oracle.pair_probability(K, xi, n, dt, dV)
        exact = Fraction(K) * xi * Fraction((n * n - n), 2) / (n // 2) * Fraction(dt) / Fraction(dV)
        assert abs(Fraction(p) - exact) <= 4 * Fraction(2) ** -53 * exact
    # the ratio is (n-1) for even n and n for odd n (R2)
    for n in range(2, 50):
        assert oracle.pair_probability(1.0, 1, n, 1.0, 1.0) == float(n - 1 if n % 2 == 0 else n)


def test_gamma_tilde_of_a_probability_that_is_not_positive():
    """DESIGN.md R20: p <= 0 or NaN (user kernel code returning a negative number or NaN) is 'no event', whatever the
    uniform and the multiplicities; the smallest positive p still fires when phi allows it, and +inf is capped by
    Eq. 4."""
    big = 10 ** 6
    for p in (float("nan"), -float("nan"), -0.3, -1.0, -7.5, -1e300, -float("inf"), -0.0, 0.0):
        for u in (0.0, 0.25, 0.999):
            for xj, xk in ((big, 1), (9, 2), (3, 3)):
                assert oracle.gamma_tilde(p, u, xj, xk) == 0, (p, u, xj, xk)
    tiny = 5e-324
    assert oracle.gamma_tilde(tiny, 0.0, big, 1) == 1 and oracle.gamma_tilde(tiny, 1e-300, big, 1) == 0
    assert oracle.gamma_tilde(float("inf"), 0.5, 9, 2) == 4
