"""GPU parity for NEXT-3, the spectrum product of Fig. 6, and the figure's content itself:
the GPU's 3600-step Golovin run at 2^20 super-droplets against Eq. 7."""
import math

import numpy as np
import pytest
from scipy import special

import oracle
import workloads

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
RHO = 1000.0


@pytest.fixture(scope="module")
def sdm_mod():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2101_06318_b200 as m
    m.load_library()
    return m


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _close(a, b, rtol=1e-12):
    return np.all(np.abs(a - b) <= rtol * np.abs(b))


def test_spectrum_matches_the_oracle_on_evolving_states(sdm_mod):
    edges, dlnr, _ = workloads.spectrum_bins(100, 2e-6, 5e-3)
    for w in (workloads.golovin_box(2 ** 15), workloads.grid_poisson(32, 32, 64.0, shuffled=True, seed=2)):
        s = sdm_mod.SDM(w.n_sd, w.n_cell)
        s.set_state(_dev(w.xi), _dev(w.v), _dev(w.cell_id))
        V = w.dV * w.n_cell
        for it in range(3):
            xi, v, _ = (t.cpu().numpy() for t in s.get_state())
            for ns in (0, 1, 2):
                got = s.spectrum(edges, dlnr, RHO, V, n_smooth=ns)
                want = oracle.spectrum(xi, v, edges, dlnr, RHO, V, n_smooth=ns)
                assert _close(got, want), (w.name, it, ns)
                assert np.array_equal(got == 0.0, want == 0.0)
            s.run(w.dt, w.dV, w.kernel, w.kparam * (1 if w.n_cell == 1 else 4000), w.seed, 40 * it, 40, True)
        s.close()


def test_spectrum_edge_cases_and_errors(sdm_mod):
    xi = np.array([3, 1, 2, 5, 1, 7, 9], dtype=np.int64)
    v = np.array([1.0, 1.5, 2.0, 3.0, 8.0, 16.0, 0.5])
    s = sdm_mod.SDM(8, 1)
    s.set_state(_dev(xi), _dev(v), _dev(np.zeros(7, dtype=np.int32)))
    edges, dlnr = np.array([1.0, 2.0, 4.0, 8.0, 16.0]), np.array([0.5, 0.5, 0.25, 0.25])
    assert s.spectrum(edges, dlnr, 2.0, 4.0, n_smooth=0).tolist() == [4.5, 19.0, 0.0, 16.0]
    assert _close(s.spectrum(edges, dlnr, 2.0, 4.0, n_smooth=2), oracle.spectrum(xi, v, edges, dlnr, 2.0, 4.0, 2), 1e-15)
    assert s.spectrum(np.array([1.0, 32.0]), np.array([1.0]), 1.0, 1.0, n_smooth=2).tolist() == [3 + 1.5 + 4 + 15 + 8 + 112]
    many = np.linspace(0.25, 20.0, 1025)
    assert _close(s.spectrum(many, np.full(1024, 0.1), 1.0, 1.0, 2), oracle.spectrum(xi, v, many, np.full(1024, 0.1), 1.0, 1.0, 2))
    for bad in ((np.array([1.0, 1.0]), np.array([1.0]), 1.0, 1.0), (np.array([1.0, 2.0]), np.array([0.0]), 1.0, 1.0),
                (np.array([1.0, 2.0]), np.array([1.0]), 0.0, 1.0), (np.array([1.0, 2.0]), np.array([1.0]), 1.0, -1.0),
                (np.linspace(1, 2, 1026), np.ones(1025), 1.0, 1.0)):
        with pytest.raises(sdm_mod.SdmError) as e:
            s.spectrum(*bad)
        assert e.value.code == -1
    s.close()


def test_fig6_golovin_spectrum_at_2e20_follows_eq7(sdm_mod):
    """Fig. 6 of the paper with 2^20 super-droplets on the GPU: mass density per ln r, ~100 bins, smoothed
    twice, at t = 1200, 2400, 3600 s against Eq. 7."""
    w = workloads.golovin_box(2 ** 20)
    s = sdm_mod.SDM(w.n_sd, w.n_cell)
    s.set_state(_dev(w.xi), _dev(w.v), _dev(w.cell_id))
    edges, dlnr, r_mid = workloads.spectrum_bins(100, 2e-6, 5e-3)
    n0, vbar, b = 2.0 ** 23, workloads.V_MEAN_BOX, w.kparam
    vol = 4.0 * math.pi / 3.0 * r_mid ** 3
    t_done = 0
    peaks = []
    for t in (1200, 2400, 3600):
        s.run(w.dt, w.dV, w.kernel, w.kparam, w.seed, t_done, t - t_done, True)
        t_done = t
        sm = s.spectrum(edges, dlnr, RHO, w.dV, n_smooth=2)
        tau = 1.0 - math.exp(-n0 * b * vbar * t)
        st = math.sqrt(tau)
        phi = (1 - tau) / (vol * st) * special.ive(1, 2 * vol * st / vbar) * np.exp(-vol * (1 + tau - 2 * st) / vbar)
        ana = 3.0 * RHO * vol * vol * n0 * phi
        core = ana > 0.2 * ana.max()
        assert abs(int(np.argmax(sm)) - int(np.argmax(ana))) <= 2, t
        assert np.max(np.abs(sm[core] / ana[core] - 1)) < 0.15, (t, np.max(np.abs(sm[core] / ana[core] - 1)))
        assert abs(np.sum(sm * dlnr) / (RHO * n0 * vbar) - 1) < 1e-3          # the water stays on the grid
        peaks.append(r_mid[int(np.argmax(sm))])
    assert peaks[0] < peaks[1] < peaks[2]                                    # the spectrum moves to larger radii
    s.close()
