"""Pins for the whole oracle step: hand-worked examples (P4), invariants (P5), the tie rule (R7),
compaction and moments semantics (P9).  PAPER.md:67-71, 175-218, 252-287."""
from fractions import Fraction
import math

import numpy as np

import oracle
import workloads
from conftest import read_golden


def _ints(s):
    return np.array([int(x) for x in s.split()], dtype=np.int64)


def _floats(s):
    return np.array([float(x) for x in s.split()], dtype=np.float64)


def test_handworked_keys_permutation_and_uniforms():
    g = read_golden("handworked_n4.txt")
    key64, u = oracle.rng(4, 0, 0)
    assert [int(k) for k in key64] == [int(w, 16) for w in g["key64"].split()]
    idx = oracle.permutation(np.zeros(4, dtype=np.int32), key64)
    assert idx.tolist() == _ints(g["idx"]).tolist()
    assert u[idx[0]] == float(g["u_pair0"]) and u[idx[2]] == float(g["u_pair1"])
    key2, u2 = oracle.rng(2, 0, 0)
    idx2 = oracle.permutation(np.zeros(2, dtype=np.int32), key2)
    assert idx2.tolist() == _ints(g["n2_idx"]).tolist() and u2[idx2[0]] == float(g["n2_u"])


def test_handworked_examples_A_B_C():
    g = read_golden("handworked_n4.txt")
    cell = np.zeros(4, dtype=np.int32)
    for ex in "ABC":
        xi, v = _ints(g[f"ex{ex}_xi"]), _floats(g[f"ex{ex}_v"])
        idx, cs, nev = oracle.step(xi, v, cell, 1, 1.0, 1.0, oracle.KERNEL_GOLOVIN, float(g[f"ex{ex}_b"]), 0, 0)
        assert idx.tolist() == _ints(g["idx"]).tolist() and cs.tolist() == [0, 4]
        assert xi.tolist() == _ints(g[f"ex{ex}_xi_after"]).tolist(), ex
        assert v.tolist() == _floats(g[f"ex{ex}_v_after"]).tolist(), ex
    xi2, v2, c2 = oracle.remove_zero(xi, v, cell)
    assert xi2.tolist() == _ints(g["exC_removed_xi"]).tolist()
    assert v2.tolist() == _floats(g["exC_removed_v"]).tolist() and len(c2) == 3


def test_key_ties_break_by_storage_index_and_cell_major_order():
    cell = np.array([1, 0, 1, 0, 1, 0], dtype=np.int32)
    key = np.array([5, 9, 5, 9, 1, 2], dtype=np.uint64)
    # cell 0: (2,i5) (9,i1) (9,i3) ; cell 1: (1,i4) (5,i0) (5,i2)
    assert oracle.permutation(cell, key).tolist() == [5, 1, 3, 4, 0, 2]
    # explicit storage indices decide ties, not positions
    sid = np.array([50, 40, 30, 20, 10, 0], dtype=np.int64)
    assert oracle.permutation(cell, key, sid=sid).tolist() == [5, 3, 1, 4, 2, 0]
    assert oracle.cell_start(cell, 3).tolist() == [0, 3, 6, 6]


def _total_water(xi, v):
    return sum(Fraction(int(a)) * Fraction(float(b)) for a, b in zip(xi, v))


def test_step_invariants_small_multiplicity_grid():
    w = workloads.grid_small_multiplicity(8, 8, 13, shuffled=True, seed=3)
    xi, v, cell = w.xi.copy(), w.v.copy(), w.cell_id.copy()
    n_events_total = 0
    for step in range(12):
        xi, v, cell = oracle.remove_zero(xi, v, cell)
        xi0, v0 = xi.copy(), v.copy()
        idx, cs, nev = oracle.step(xi, v, cell, w.n_cell, w.dt, w.dV, w.kernel, w.kparam, w.seed, step)
        n_events_total += nev
        n = len(xi)
        assert sorted(idx.tolist()) == list(range(n))                       # a permutation
        assert np.all(np.diff(cell[idx]) >= 0)                              # cell-major
        assert np.array_equal(cs, np.concatenate([[0], np.cumsum(np.bincount(cell, minlength=w.n_cell))]))
        key64, _ = oracle.rng(n, w.seed, step)
        for c in range(w.n_cell):
            seg = idx[cs[c]:cs[c + 1]]
            assert np.all(np.diff(key64[seg].astype(object)) >= 0)          # keys ascending in a cell
        assert np.all(xi >= 0) and np.all(v >= v0)                          # v never decreases
        assert xi.sum() <= xi0.sum()                                        # sum xi monotone
        # v takes integer values here, so water is conserved exactly
        assert _total_water(xi, v) == _total_water(xi0, v0)
        # at most the two members of a pair change; changes come in pairs (2m, 2m+1) of a cell
        changed = set(np.nonzero((xi != xi0) | (v != v0))[0].tolist())
        pos = {int(d): p for p, d in enumerate(idx)}
        for d in changed:
            p = pos[d]
            c = cell[d]
            m = (p - cs[c]) // 2
            assert cs[c] + 2 * m + 1 < cs[c + 1]                            # the odd one out never changes
        assert len(changed) <= 2 * nev
    assert n_events_total > 100 and len(xi) < w.n_sd                        # the case really collides/removes


def test_sum_xi_decrease_equals_sum_of_g_xi_k():
    # exact int64 bookkeeping on a box with big multiplicities: every event removes g*xi_k
    w = workloads.golovin_box(2 ** 10)
    xi, v = w.xi.copy(), w.v.copy()
    for step in range(50):
        xi0 = xi.copy()
        idx, cs, nev = oracle.step(xi, v, w.cell_id, 1, w.dt, w.dV, w.kernel, w.kparam, 0, step)
        dec = 0
        for m in range(len(xi) // 2):
            a, b = idx[2 * m], idx[2 * m + 1]
            if xi[a] != xi0[a] or xi[b] != xi0[b]:
                j, k = (a, b) if xi0[a] >= xi0[b] else (b, a)
                if xi[k] == xi0[k]:
                    assert (xi0[j] - xi[j]) % xi0[k] == 0                   # Eq. 5: g * xi_k
                else:
                    assert xi[j] + xi[k] == xi0[k]                          # Eq. 6: split of xi_k
                dec += (xi0[a] + xi0[b]) - (xi[a] + xi[b])
        assert xi0.sum() - xi.sum() == dec


def test_odd_cells_and_tiny_cells():
    cell = np.array([0, 2, 2, 2, 3], dtype=np.int32)          # cell 1 empty, cells 0 and 3 single
    xi = np.array([5, 5, 5, 5, 5], dtype=np.int64)
    v = np.ones(5)
    idx, cs, nev = oracle.step(xi, v, cell, 4, 1.0, 1.0, 0, 1e6, 1, 1)   # p huge -> every pair fires
    assert cs.tolist() == [0, 1, 1, 4, 5] and nev == 1
    unpaired = idx[3]                                          # third of the 3-droplet cell
    assert xi[0] == 5 and xi[4] == 5 and xi[unpaired] == 5
    assert sorted(xi[idx[1:3]].tolist()) == [2, 3]


def test_remove_zero_is_a_stable_filter():
    rng = np.random.default_rng(0)
    xi = rng.integers(0, 3, 1000).astype(np.int64)
    v = rng.random(1000)
    cell = rng.integers(0, 7, 1000).astype(np.int32)
    a, b, c = oracle.remove_zero(xi, v, cell)
    keep = xi != 0
    assert np.array_equal(a, xi[keep]) and np.array_equal(b, v[keep]) and np.array_equal(c, cell[keep])
    e = oracle.remove_zero(np.zeros(5, dtype=np.int64), np.ones(5), np.zeros(5, dtype=np.int32))
    assert all(len(x) == 0 for x in e)


def test_moments_against_exact_sums():
    rng = np.random.default_rng(1)
    n, n_cell = 5000, 9
    xi = rng.integers(0, 10 ** 9, n).astype(np.int64)
    v = np.exp(rng.normal(-30, 3, n))
    cell = rng.integers(0, n_cell, n).astype(np.int32)
    m0, m1, m2 = oracle.moments(xi, v)
    assert m0 == int(xi.sum())
    assert m1 == math.fsum(float(a) * b for a, b in zip(xi, v))
    assert m2 == math.fsum((float(a) * b) * b for a, b in zip(xi, v))
    p0, p1, p2 = oracle.moments(xi, v, cell, n_cell, per_cell=True)
    for c in range(n_cell):
        sel = cell == c
        assert p0[c] == int(xi[sel].sum())
        assert p1[c] == math.fsum(float(a) * b for a, b in zip(xi[sel], v[sel]))
        assert p2[c] == math.fsum((float(a) * b) * b for a, b in zip(xi[sel], v[sel]))
    # exact rational cross-check of M1 on a short prefix
    exact = sum(Fraction(int(a)) * Fraction(float(b)) for a, b in zip(xi[:200], v[:200]))
    assert abs(Fraction(oracle.moments(xi[:200].copy(), v[:200].copy())[1]) - exact) < Fraction(1, 10 ** 13) * exact


def test_subset_with_storage_indices_reproduces_full_step():
    # cells are independent: running the oracle on one cell's droplets with their global storage
    # indices gives the same result as the full step (used for sampled parity at full size)
    w = workloads.grid_small_multiplicity(6, 6, 10, shuffled=True, seed=5)
    xi, v = w.xi.copy(), w.v.copy()
    idx, cs, _ = oracle.step(xi, v, w.cell_id, w.n_cell, w.dt, w.dV, w.kernel, w.kparam, 9, 4)
    for c in (0, 7, 35):
        sel = np.nonzero(w.cell_id == c)[0]
        xs, vs = w.xi[sel].copy(), w.v[sel].copy()
        li, _, _ = oracle.step(xs, vs, np.zeros(len(sel), dtype=np.int32), 1, w.dt, w.dV, w.kernel,
                               w.kparam, 9, 4, sid=sel.astype(np.int64))
        assert np.array_equal(sel[li], idx[cs[c]:cs[c + 1]])
        assert np.array_equal(xs, xi[sel]) and np.array_equal(vs, v[sel])
