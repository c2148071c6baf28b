"""Pins for the coalescence kernels of the oracle (row a5): Golovin, the
gravitational kernel of BASELINE.json config 3 and the specified cube root (R9, R10)."""
from fractions import Fraction
import math

import numpy as np

import oracle
from conftest import read_golden

C34PI = 3.0 / (4.0 * math.pi)


def _vol(r):
    return 4.0 * math.pi / 3.0 * r ** 3


def test_cbrt_spec_within_one_ulp_exact_rational_check():
    rng = np.random.default_rng(0)
    xs = np.exp(rng.uniform(math.log(1e-40), math.log(1e20), 4000))
    xs = np.concatenate([xs, [1.0, 8.0, 27.0, 1e-15, 2.0 ** -300, 2.0 ** 300, 0.238732414637843e-14]])
    for x in xs:
        x = float(x)
        r = oracle.cbrt_spec(x)
        ulp = float(np.spacing(r))
        lo, hi = Fraction(r) - Fraction(ulp), Fraction(r) + Fraction(ulp)
        assert lo ** 3 < Fraction(x) < hi ** 3, x
    assert oracle.cbrt_spec(27.0) == 3.0 and oracle.cbrt_spec(1.0) == 1.0


def test_cbrt_spec_close_to_libm():
    xs = np.exp(np.random.default_rng(1).uniform(math.log(1e-25), math.log(1e-5), 20000))
    r = np.array([oracle.cbrt_spec(float(x)) for x in xs])
    assert np.max(np.abs(r - np.cbrt(xs)) / np.spacing(np.cbrt(xs))) <= 2.0


def test_golovin_kernel():
    assert oracle.kernel(oracle.KERNEL_GOLOVIN, 1500.0, 2.0, 3.0) == 7500.0
    assert oracle.kernel(oracle.KERNEL_GOLOVIN, 1500.0, 1e-13, 3e-13) == 1500.0 * (1e-13 + 3e-13)


def test_gravitational_kernel_hand_values():
    g = read_golden("gravitational_kernel.txt")
    for case in "ABC":
        r1, r2 = float(g[f"case{case}_r1"]), float(g[f"case{case}_r2"])
        K = oracle.kernel(oracle.KERNEL_GRAVITATIONAL, 1.0, _vol(r1), _vol(r2))
        want = math.pi * float(g[f"case{case}_K_over_pi"])
        assert abs(K - want) <= 1e-12 * want
        # symmetric, exactly; E scales linearly
        assert K == oracle.kernel(oracle.KERNEL_GRAVITATIONAL, 1.0, _vol(r2), _vol(r1))
        # E enters as one factor: a power of two scales K exactly
        assert oracle.kernel(oracle.KERNEL_GRAVITATIONAL, 0.5, _vol(r1), _vol(r2)) == 0.5 * K
    assert oracle.kernel(oracle.KERNEL_GRAVITATIONAL, 1.0, _vol(30e-6), _vol(30e-6)) == 0.0


def _w_via_kernel(r):
    """Terminal velocity recovered from K against a vanishing partner (r2 = 1e-10 m, w2 ~ 1e-12)."""
    r2 = 1e-10
    K = oracle.kernel(oracle.KERNEL_GRAVITATIONAL, 1.0, _vol(r), _vol(r2))
    return K / (math.pi * (r + r2) ** 2) + 1.19e8 * r2 * r2


def test_terminal_velocity_regime_joins():
    g = read_golden("gravitational_kernel.txt")
    below40 = float(np.nextafter(40e-6, 0) * (1 - 1e-9))
    assert abs(_w_via_kernel(below40) - float(g["w_below_40um"])) < 1e-6
    assert abs(_w_via_kernel(40e-6 * (1 + 1e-9)) - float(g["w_at_40um"])) < 1e-6
    assert abs(_w_via_kernel(600e-6 * (1 - 1e-9)) - float(g["w_below_600um"])) < 1e-5
    assert abs(_w_via_kernel(600e-6 * (1 + 1e-9)) - float(g["w_at_600um"])) < 1e-5


# ---- NEXT-2: tabulated collection efficiency (R16) ----------------

_GRID = np.array([10e-6, 20e-6, 40e-6])
_ETAB = np.array([[0.0, 0.1, 0.2], [0.1, 0.4, 0.6], [0.2, 0.6, 1.0]])


def test_efficiency_table_hand_values_and_clamping():
    g = read_golden("efficiency_table.txt")
    oracle.set_efficiency_table(_GRID, _ETAB)
    for key, (r1, r2) in {"E_15_20": (15e-6, 20e-6), "E_15_30": (15e-6, 30e-6), "E_25_35": (25e-6, 35e-6),
                          "E_5_5": (5e-6, 5e-6), "E_80_80": (80e-6, 80e-6), "E_5_80": (5e-6, 80e-6)}.items():
        assert abs(oracle.efficiency(r1, r2) - float(g[key])) <= 1e-12, key
        assert abs(oracle.efficiency(r1, r2) - oracle.efficiency(r2, r1)) <= 1e-15   # symmetric table
    # grid nodes reproduce the table exactly
    for i, ri in enumerate(_GRID):
        for k, rk in enumerate(_GRID):
            assert oracle.efficiency(float(ri), float(rk)) == _ETAB[i, k]
    # bilinear interpolation of a function that IS bilinear is exact up to rounding: E = a + b r1 + c r2 + d r1 r2
    grid = np.array([1.0, 2.0, 4.0, 8.0])
    f = lambda x, y: 0.5 + 0.25 * x + 0.125 * y + 0.0625 * x * y
    oracle.set_efficiency_table(grid, f(grid[:, None], grid[None, :]))
    rng = np.random.default_rng(3)
    for x, y in rng.uniform(1.0, 8.0, (300, 2)):
        assert abs(oracle.efficiency(x, y) - f(x, y)) <= 1e-13 * f(x, y)


def test_efficiency_table_validation():
    for grid, tab in ((np.array([1.0]), np.ones((1, 1))), (np.array([2.0, 1.0]), np.ones((2, 2))),
                      (np.array([1.0, 1.0]), np.ones((2, 2))), (np.array([1.0, 2.0]), -np.ones((2, 2))),
                      (np.array([1.0, 2.0]), np.full((2, 2), np.nan)), (np.array([0.0, 2.0]), np.ones((2, 2)))):
        try:
            oracle.set_efficiency_table(grid, tab)
        except ValueError:
            continue
        raise AssertionError("invalid table accepted")


def test_tabulated_kernel_reduces_to_the_gravitational_kernel_and_scales_with_the_table():
    rng = np.random.default_rng(5)
    vs = _vol(np.exp(rng.uniform(math.log(2e-6), math.log(2e-3), (200, 2))))
    oracle.set_efficiency_table(_GRID, np.ones((3, 3)))                          # E == 1: the plain kernel, bit for bit
    for vj, vk in vs:
        assert (oracle.kernel(oracle.KERNEL_GRAVITATIONAL_TABULATED, 0.75, vj, vk)
                == oracle.kernel(oracle.KERNEL_GRAVITATIONAL, 0.75, vj, vk))
    oracle.set_efficiency_table(_GRID, _ETAB)
    for vj, vk in vs:
        rj, rk = oracle.cbrt_spec(vj * C34PI), oracle.cbrt_spec(vk * C34PI)
        K1 = oracle.kernel(oracle.KERNEL_GRAVITATIONAL, 1.0, vj, vk)
        K2 = oracle.kernel(oracle.KERNEL_GRAVITATIONAL_TABULATED, 1.0, vj, vk)
        assert abs(K2 - oracle.efficiency(rj, rk) * K1) <= 1e-14 * K1
        # interpolating along r_j first is not bit-symmetric; the step always passes (j, k) in a defined order
        assert abs(K2 - oracle.kernel(oracle.KERNEL_GRAVITATIONAL_TABULATED, 1.0, vk, vj)) <= 4e-16 * K2
