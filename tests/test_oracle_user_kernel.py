"""Oracle pins for NEXT-2's user-supplied kernel code: ORC_KERNEL_USER calls a C function the
caller supplies.  What is pinned is the CONTRACT of the hook, not the user's formula: which volume arrives as v_j, that
the parameters arrive in order, that nothing else changes (a built-in kernel re-expressed as user code reproduces the
built-in step bit for bit), and the value Eq. 3 receives (hand-worked outcome on two droplets)."""
import numpy as np

import oracle
import workloads

GOLOVIN_C = "double sdm_user_kernel(double vj, double vk, const double *p) { double s = vj + vk; return p[0] * s; }"


def test_golovin_as_user_code_reproduces_the_builtin_step_bit_for_bit():
    w = workloads.grid_small_multiplicity(6, 6, 24, seed=9)
    oracle.set_user_kernel(GOLOVIN_C, [w.kparam])
    a = (w.xi.copy(), w.v.copy())
    b = (w.xi.copy(), w.v.copy())
    ev_a = ev_b = 0
    for step in range(5):
        ev_a += oracle.step(a[0], a[1], w.cell_id, w.n_cell, w.dt, w.dV, oracle.KERNEL_GOLOVIN, w.kparam, 3, step)[2]
        ev_b += oracle.step(b[0], b[1], w.cell_id, w.n_cell, w.dt, w.dV, oracle.KERNEL_USER, 0.0, 3, step)[2]
    assert ev_a == ev_b > 100
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_parameters_arrive_in_order_and_products_are_not_contracted():
    # a = p0*vj + p1*vk, every product and the sum rounded separately (gcc -ffp-contract=off)
    oracle.set_user_kernel("double sdm_user_kernel(double vj, double vk, const double *p) { return p[0] * vj + p[1] * vk; }",
                           [0.1, 3.0])
    vj, vk = 1.0 / 3.0, 1e-17
    assert oracle.kernel(oracle.KERNEL_USER, 0.0, vj, vk) == (0.1 * vj) + (3.0 * vk)


def test_vj_is_the_volume_of_the_larger_multiplicity_hand_worked():
    """Two droplets, xi = (2, 5), v = (1, 1000): j is droplet 1 (Fig. 5).  Kernel = 1 if vj > vk else 0.
    With dt = dV = 1: p = 1 * 5 * 1 = 5 > 1, so gamma = 5 whatever the uniform, capped at floor(5/2) = 2 (Eq. 4):
    xi_1 = 5 - 2*2 = 1, v_0 = 1 + 2*1000 (Eq. 5).  Had the arguments been swapped, K = 0 and nothing would change."""
    oracle.set_user_kernel("double sdm_user_kernel(double vj, double vk, const double *p) { return vj > vk ? 1.0 : 0.0; }")
    xi, v = np.array([2, 5], dtype=np.int64), np.array([1.0, 1000.0])
    _, _, nev = oracle.step(xi, v, np.zeros(2, dtype=np.int32), 1, 1.0, 1.0, oracle.KERNEL_USER, 0.0, 0, 0)
    assert nev == 1 and xi.tolist() == [2, 1] and v.tolist() == [2001.0, 1000.0]
    # mirrored state: now droplet 0 is j, and v_j = 1 < v_k: K = 0, no event
    xi, v = np.array([5, 2], dtype=np.int64), np.array([1.0, 1000.0])
    _, _, nev = oracle.step(xi, v, np.zeros(2, dtype=np.int32), 1, 1.0, 1.0, oracle.KERNEL_USER, 0.0, 0, 0)
    assert nev == 0 and xi.tolist() == [5, 2]


def test_negative_and_nan_kernel_values_leave_the_pair_alone():
    """DESIGN.md R20 through a whole step: user code that returns a negative number or NaN for some pairs produces no
    event there -- the same two droplets as above, so the outcome is known by hand.  A negative value with the old
    arithmetic gave gamma = -1 or 0 and xi_j = 5 + 2 = 7 (multiplicities growing); NaN reached an int64 cast."""
    for body in ("return -1.0;", "double z = vj - vj; return z / z;", "return vj > vk ? -0.25 : 3.0;"):
        oracle.set_user_kernel("double sdm_user_kernel(double vj, double vk, const double *p) { " + body + " }")
        for seed in range(20):                      # whatever the uniform
            xi, v = np.array([2, 5], dtype=np.int64), np.array([1.0, 1000.0])
            _, _, nev = oracle.step(xi, v, np.zeros(2, dtype=np.int32), 1, 1.0, 1.0, oracle.KERNEL_USER, 0.0, seed, 0)
            assert nev == 0 and xi.tolist() == [2, 5] and v.tolist() == [1.0, 1000.0], (body, seed)
    # the third kernel is positive for the mirrored order (v_j = 1 < v_k = 1000): p = 3 * 5 = 15, cap floor(5/2) = 2
    xi, v = np.array([5, 2], dtype=np.int64), np.array([1.0, 1000.0])
    _, _, nev = oracle.step(xi, v, np.zeros(2, dtype=np.int32), 1, 1.0, 1.0, oracle.KERNEL_USER, 0.0, 0, 0)
    assert nev == 1 and xi.tolist() == [1, 2] and v.tolist() == [1.0, 1002.0]
