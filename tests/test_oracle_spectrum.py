"""Pins of the oracle's spectrum product (Fig. 6 and Eq. 7)."""
import math

import numpy as np
from scipy import special

import oracle
import workloads
from conftest import read_golden

RHO = 1000.0          # "assuming particle density of 1000 kg/m^3"


def test_hand_worked_bins_and_smoothing():
    g = read_golden("spectrum_product.txt")
    xi = np.array([3, 1, 2, 5, 1, 7, 9], dtype=np.int64)
    v = np.array([1.0, 1.5, 2.0, 3.0, 8.0, 16.0, 0.5])
    edges = np.array([1.0, 2.0, 4.0, 8.0, 16.0])
    dlnr = np.array([0.5, 0.5, 0.25, 0.25])
    for key, ns in (("raw", 0), ("smooth1", 1), ("smooth2", 2)):
        want = np.array([float(x) for x in g[key].split()])
        got = oracle.spectrum(xi, v, edges, dlnr, 2.0, 4.0, n_smooth=ns)
        assert np.allclose(got, want, rtol=1e-15, atol=0), (key, got)


def test_unsmoothed_spectrum_conserves_the_binned_mass_and_smoothing_stays_within_bounds():
    rng = np.random.default_rng(0)
    n = 20000
    xi = rng.integers(1, 1000, n).astype(np.int64)
    v = np.exp(rng.uniform(math.log(1e-16), math.log(1e-9), n))
    edges, dlnr, _ = workloads.spectrum_bins(60, 1e-6, 1e-3)
    raw = oracle.spectrum(xi, v, edges, dlnr, RHO, 7.0, n_smooth=0)
    inside = (v >= edges[0]) & (v < edges[-1])
    mass = math.fsum((xi[inside] * v[inside]).tolist()) * RHO / 7.0
    assert abs(float(np.sum(raw * dlnr)) - mass) <= 1e-12 * mass
    # bin membership against numpy's own search
    b = np.searchsorted(edges, v[inside], side="right") - 1
    ref = np.zeros(60)
    np.add.at(ref, b, xi[inside] * v[inside])
    assert np.allclose(raw, ref * RHO / 7.0 / dlnr, rtol=1e-12, atol=0)
    # the running mean with truncated windows keeps every value between the extremes of the raw spectrum
    sm = oracle.spectrum(xi, v, edges, dlnr, RHO, 7.0, n_smooth=2)
    assert raw.min() <= sm.min() and sm.max() <= raw.max()


def _golovin_mass_density(r, t, n0, vbar, b):
    """Eq. 7 as mass per unit ln r: 3 rho v^2 N0 phi(v, t)."""
    v = 4.0 * math.pi / 3.0 * r ** 3
    tau = 1.0 - math.exp(-n0 * b * vbar * t)
    if tau == 0.0:
        phi = np.exp(-v / vbar) / vbar
    else:
        st = math.sqrt(tau)
        phi = (1 - tau) / (v * st) * special.ive(1, 2 * v * st / vbar) * np.exp(-v * (1 + tau - 2 * st) / vbar)
    return 3.0 * RHO * v * v * n0 * phi


def test_initial_box_spectrum_matches_the_exponential_distribution():
    # t = 0: phi = exp(-v/vbar)/vbar; per bin the exact mass is N0 [-(v + vbar) exp(-v/vbar)] over the bin
    w = workloads.golovin_box(2 ** 17)
    edges, dlnr, r_mid = workloads.spectrum_bins(100, 2e-6, 2e-3)
    raw = oracle.spectrum(w.xi, w.v, edges, dlnr, RHO, w.dV, n_smooth=0)
    n0, vbar = 2.0 ** 23, workloads.V_MEAN_BOX
    F = lambda x: -(x + vbar) * np.exp(-x / vbar)
    exact = RHO * n0 * (F(edges[1:]) - F(edges[:-1])) / dlnr
    big = exact > 0.1 * exact.max()           # the far tail is cut by the 99.999 % quantile
    assert big.sum() > 15
    assert np.max(np.abs(raw[big] / exact[big] - 1)) < 0.01          # quantile discretisation with 2^17 droplets
    assert abs(np.sum(raw * dlnr) / (RHO * n0 * vbar) - 1) < 1e-3     # all the water is inside the grid
    # and Eq. 7 at t = 0 is that density
    assert np.max(np.abs(_golovin_mass_density(r_mid[big], 0.0, n0, vbar, 1500.0) / exact[big] - 1)) < 0.03   # point value at the bin centre vs bin average


def test_smoothed_spectrum_follows_eq7_after_1200_s():
    # Fig. 6 of the paper at reduced size: 2^14 droplets, 1200 steps, binned and smoothed twice
    w = workloads.golovin_box(2 ** 14)
    xi, v, cell = w.xi.copy(), w.v.copy(), w.cell_id.copy()
    for step in range(1200):
        xi, v, cell = oracle.remove_zero(xi, v, cell)
        oracle.step(xi, v, cell, 1, w.dt, w.dV, w.kernel, w.kparam, w.seed, step, want_perm=False)
    edges, dlnr, r_mid = workloads.spectrum_bins(100, 2e-6, 5e-3)
    sm = oracle.spectrum(xi, v, edges, dlnr, RHO, w.dV, n_smooth=2)
    ana = _golovin_mass_density(r_mid, 1200.0, 2.0 ** 23, workloads.V_MEAN_BOX, w.kparam)
    # the position of the mass peak moved from ~ 45 um to ~ 100 um and agrees within a bin or two
    assert abs(int(np.argmax(sm)) - int(np.argmax(ana))) <= 3
    assert 60e-6 < r_mid[int(np.argmax(sm))] < 200e-6
    core = ana > 0.2 * ana.max()
    assert np.max(np.abs(sm[core] / ana[core] - 1)) < 0.35            # Monte-Carlo noise of 2^14 droplets
    assert abs(np.sum(sm * dlnr) / np.sum(ana * dlnr) - 1) < 0.05
