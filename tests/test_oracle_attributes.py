"""Pins of the oracle's multi-attribute update: the loop over extensive attributes
of Fig. 5 on the 2-D row-major attribute block of Fig. 2."""
import numpy as np

import oracle
import workloads
from conftest import read_golden


def test_paper_worked_example_with_two_attributes():
    g = read_golden("paper_worked_examples.txt")
    xi = np.array([9, 2], dtype=np.int64)
    attr = np.array([[3.0, 7.0], [10.0, 0.5]])
    oracle.collide_pair_attr(xi, attr, 0, 1, 5)                       # gamma = 5 -> gamma_tilde = 4
    assert xi.tolist() == [1, 2]
    assert attr[0].tolist() == [3.0, float(g["fig1b_attr_A_k_after"])]
    assert attr[1].tolist() == [10.0, float(g["fig1b_attr_B_k_after"])]
    # stored the other way round: j is still the droplet with the larger multiplicity
    xi = np.array([2, 9], dtype=np.int64)
    attr = np.array([[7.0, 3.0], [0.5, 10.0]])
    oracle.collide_pair_attr(xi, attr, 0, 1, 5)
    assert xi.tolist() == [2, 1] and attr[0].tolist() == [19.0, 3.0] and attr[1].tolist() == [40.5, 10.0]
    # Eq. 6: equal multiplicities, both droplets carry g*A_j + A_k in every row
    xi = np.array([4, 4], dtype=np.int64)
    attr = np.array([[3.0, 7.0], [10.0, 0.5]])
    oracle.collide_pair_attr(xi, attr, 0, 1, 1)
    assert xi.tolist() == [2, 2]
    assert attr[0].tolist() == [float(g["eq6_attr_A_after"])] * 2
    assert attr[1].tolist() == [float(g["eq6_attr_B_after"])] * 2


def _small_state(seed, n_attr):
    w = workloads.grid_small_multiplicity(8, 8, 24, seed=seed, shuffled=True)
    rng = np.random.default_rng(seed + 100)
    attr = np.empty((n_attr, w.n_sd))
    attr[0] = w.v
    for r in range(1, n_attr):
        attr[r] = rng.integers(1, 50, w.n_sd).astype(np.float64)        # small integers: sums stay exact in fp64
    return w, attr


def test_row_zero_is_the_single_attribute_step_and_rows_do_not_interact():
    w, attr = _small_state(3, 3)
    xi_a, xi_b = w.xi.copy(), w.xi.copy()
    v = w.v.copy()
    for step in range(6):
        ia, ca, ea = oracle.step_attr(xi_a, attr, w.cell_id, w.n_cell, w.dt, w.dV, w.kernel, w.kparam, 9, step)
        ib, cb, eb = oracle.step(xi_b, v, w.cell_id, w.n_cell, w.dt, w.dV, w.kernel, w.kparam, 9, step)
        assert ea == eb > 0 and np.array_equal(ia, ib) and np.array_equal(ca, cb)
        assert np.array_equal(xi_a, xi_b) and np.array_equal(attr[0], v)


def test_every_extensive_attribute_is_conserved_exactly_and_a_copy_of_the_volume_stays_a_copy():
    # Eqs. 5-6 conserve sum xi*A for every extensive attribute; with small-integer
    # values all products and sums are exact in fp64, so conservation is exact.  A row that starts as a
    # copy of row 0 undergoes the same operations and must stay bit-identical.
    w, attr = _small_state(5, 4)
    attr[3] = attr[0]
    xi, cell = w.xi.copy(), w.cell_id.copy()
    tot = [int(np.sum(xi * attr[r].astype(np.int64))) for r in range(3)]
    n_removed = 0
    for step in range(12):
        xi, attr, cell = oracle.remove_zero_attr(xi, attr, cell)
        n_removed = w.n_sd - len(xi)
        oracle.step_attr(xi, attr, cell, w.n_cell, w.dt, w.dV, w.kernel, w.kparam, 1, step, want_perm=False)
        assert np.array_equal(attr[3], attr[0])
        for r in range(3):
            assert np.all(attr[r] == np.floor(attr[r]))
            assert int(np.sum(xi * attr[r].astype(np.int64))) == tot[r], (step, r)
    assert n_removed > 0


def test_remove_zero_attr_is_a_stable_filter_of_every_row():
    rng = np.random.default_rng(2)
    n = 500
    xi = rng.integers(0, 3, n).astype(np.int64)
    attr = rng.random((3, n))
    cell = rng.integers(0, 9, n).astype(np.int32)
    keep = xi != 0
    x2, a2, c2 = oracle.remove_zero_attr(xi, attr, cell)
    assert np.array_equal(x2, xi[keep]) and np.array_equal(c2, cell[keep]) and np.array_equal(a2, attr[:, keep])
