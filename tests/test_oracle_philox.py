"""Pins for the oracle's RNG step (a1): Philox4x32-10 known answers and stream conventions.
PAPER.md:186, 212 (urand), 102 (phi ~ U[0,1)); R6."""
import numpy as np
from scipy import stats

import oracle
from conftest import read_golden


def _words(s):
    return [int(w, 16) for w in s.split()]


def test_known_answer_vectors():
    g = read_golden("philox4x32_10_kat.txt")
    for k in range(3):
        out = oracle.philox4x32_10(_words(g[f"kat{k}_ctr"]), _words(g[f"kat{k}_key"]))
        assert [int(x) for x in out] == _words(g[f"kat{k}_out"])


def test_stream_layout_counter_is_storage_index_and_step():
    # block for droplet i at (seed, step) is Philox(ctr={i lo, i hi, step lo, step hi}, key={seed lo, seed hi})
    seed, step = 0x0123456789ABCDEF, 0xFEDCBA9876543210
    sid = np.array([0, 1, 5, 2 ** 32 + 7, 2 ** 40], dtype=np.int64)
    key64, u = oracle.rng(len(sid), seed, step, sid=sid)
    for n, s in enumerate(sid):
        s = int(s)
        w = oracle.philox4x32_10([s & 0xFFFFFFFF, s >> 32, step & 0xFFFFFFFF, step >> 32],
                                 [seed & 0xFFFFFFFF, seed >> 32])
        w = [int(x) for x in w]
        assert int(key64[n]) == w[0] | (w[1] << 32)
        bits = w[2] | (w[3] << 32)
        assert u[n] == (bits >> 11) / 2.0 ** 53
        assert 0.0 <= u[n] < 1.0


def test_first_block_matches_published_vector():
    # seed 0, step 0, droplet 0 is exactly the all-zero known answer
    key64, u = oracle.rng(1, 0, 0)
    assert int(key64[0]) == 0xE169C58D6627E8D5
    assert u[0] == ((0xBC57AC4C | (0x9B00DBD8 << 32)) >> 11) / 2.0 ** 53


def test_identity_sid_equals_explicit_sid():
    k0, u0 = oracle.rng(1000, 3, 9)
    k1, u1 = oracle.rng(1000, 3, 9, sid=np.arange(1000, dtype=np.int64))
    assert np.array_equal(k0, k1) and np.array_equal(u0, u1)


def test_uniformity_of_u_and_keys():
    key64, u = oracle.rng(200_000, 7, 11)
    assert stats.kstest(u, "uniform").pvalue > 1e-4
    kk = (key64 >> np.uint64(11)).astype(np.float64) / 2.0 ** 53
    assert stats.kstest(kk, "uniform").pvalue > 1e-4
    # keys and uniforms of the same droplet are uncorrelated; consecutive steps decorrelate
    assert abs(np.corrcoef(u, kk)[0, 1]) < 0.01
    _, u2 = oracle.rng(200_000, 7, 12)
    assert abs(np.corrcoef(u, u2)[0, 1]) < 0.01


def test_argsort_of_keys_is_uniform_over_orders():
    # P8: argsort of iid 64-bit keys is uniform over the n! orders (n = 3: 6 orders)
    counts = {}
    trials = 12000
    cell = np.zeros(3, dtype=np.int32)
    for step in range(trials):
        key64, _ = oracle.rng(3, 42, step)
        idx = tuple(int(i) for i in oracle.permutation(cell, key64))
        counts[idx] = counts.get(idx, 0) + 1
    assert len(counts) == 6
    chi2 = sum((c - trials / 6) ** 2 / (trials / 6) for c in counts.values())
    assert chi2 < stats.chi2.ppf(1 - 1e-4, 5)
