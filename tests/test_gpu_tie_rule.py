"""The tie rule of the per-cell permutation on the DEVICE (R7: equal sort keys are broken by storage index).
Philox output never produces equal 64-bit keys, so the kernels' equal-key and truncated-key branches are driven with
hand-made keys through sdm_debug_permutation, which runs rows a2-a3 of a step through the very kernels a real step of
the state would take.  The expected order is the oracle's argsort by (cell, key64, storage index), itself pinned on the
CPU with hand-made keys (tests/test_oracle_step.py)."""
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


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _keys(n, kind, rng):
    """Hand-made key sets that a hash never produces."""
    if kind == "all_equal":
        return np.full(n, 0x0123456789ABCDEF, dtype=np.uint64)
    if kind == "few_values":            # long runs of EQUAL key64: order inside a run = storage index
        vals = np.array([0, 1, 1 << 40, (1 << 63) + 5, 0xFFFFFFFFFFFFFFFF], dtype=np.uint64)
        return vals[rng.integers(0, len(vals), n)]
    if kind == "low_bits":              # equal top 24/32 bits, different low bits: the truncated-key branches
        hi = np.array([0x00000001, 0x7FFFFFFF, 0xABCDEF01], dtype=np.uint64)[rng.integers(0, 3, n)]
        return (hi << np.uint64(32)) | rng.integers(0, 4, n).astype(np.uint64)
    if kind == "mixed":                 # random keys with a third of them duplicated
        k = rng.integers(0, 1 << 62, n).astype(np.uint64) << np.uint64(2)
        dup = rng.random(n) < 0.33
        k[dup] = k[rng.integers(0, n, int(dup.sum()))]
        return k
    raise ValueError(kind)


def _check(sdm_mod, counts, shuffled, kind, options=(), expect_mode=None, seed=0):
    rng = np.random.default_rng(seed)
    counts = np.asarray(counts)
    cell = np.repeat(np.arange(len(counts), dtype=np.int32), counts)
    n = len(cell)
    if shuffled:
        cell = np.ascontiguousarray(cell[rng.permutation(n)])
    keys = _keys(n, kind, rng)
    s = sdm_mod.SDM(max(n, 1), len(counts))
    for k, val in options:
        s.set_option(k, val)
    xi = rng.integers(1, 9, n).astype(np.int64)
    v = rng.uniform(0.5, 2.0, n)
    s.set_state(_dev(xi), _dev(v), _dev(cell))
    if expect_mode is not None:
        assert s.counters()["mode"] == expect_mode
    s.debug_permutation(_dev(keys.view(np.int64)))
    gidx, gcs = (t.cpu().numpy() for t in s.get_permutation(n))
    want = oracle.permutation(cell, keys)
    assert np.array_equal(gcs, oracle.cell_start(cell, len(counts)))
    assert np.array_equal(gidx, want), f"{kind}: first difference at {np.nonzero(gidx != want)[0][:5]}"
    gxi, gv, _ = (t.cpu().numpy() for t in s.get_state())
    assert np.array_equal(gxi, xi) and np.array_equal(gv, v)          # no pair was evaluated
    # a real step afterwards is unaffected by the hook
    w = workloads.Workload("t", xi, v, cell, len(counts), 1.0, 1.0, 0, 0.01, 0, seed=3)
    idx, _, _ = oracle.step(xi, v, cell, w.n_cell, 1.0, 1.0, 0, 0.01, 3, 0)
    s.coalescence_step(1.0, 1.0, 0, 0.01, 3, 0)
    assert np.array_equal(s.get_permutation(n)[0].cpu().numpy(), idx)
    assert np.array_equal(s.get_state()[0].cpu().numpy(), xi)
    s.close()


KINDS = ["all_equal", "few_values", "low_bits", "mixed"]


@pytest.mark.parametrize("kind", KINDS)
def test_counting_sort_kernel_cells_up_to_256(sdm_mod, kind):
    _check(sdm_mod, [256, 256, 0, 255, 1, 130, 256, 256, 256, 7, 200], False, kind, expect_mode=1, seed=1)


@pytest.mark.parametrize("kind", KINDS)
def test_register_network_kernels(sdm_mod, kind):
    _check(sdm_mod, [64, 3, 0, 61, 1, 40], False, kind, options=[(sdm_mod.OPT_SORT_ENGINE, 1)], expect_mode=1, seed=2)
    _check(sdm_mod, [128, 99, 2, 0, 77], False, kind, options=[(sdm_mod.OPT_SORT_ENGINE, 1)], expect_mode=1, seed=3)
    _check(sdm_mod, [400, 512, 3, 300], False, kind, expect_mode=1, seed=4)


@pytest.mark.parametrize("kind", KINDS)
def test_general_path_cells_and_split_cells(sdm_mod, kind):
    _check(sdm_mod, [100, 256, 0, 1, 37, 255], True, kind, expect_mode=0, seed=5)
    # cells larger than a segment are cut by the top key bits: with hand-made keys whole cells land in one bucket,
    # far beyond the segment capacity (the ranking-by-counting fallback)
    _check(sdm_mod, [700, 5, 1300], True, kind, expect_mode=0, seed=6)


@pytest.mark.parametrize("kind", KINDS)
def test_box_path(sdm_mod, kind):
    _check(sdm_mod, [3000], False, kind, expect_mode=2, seed=7)
    _check(sdm_mod, [2], False, kind, expect_mode=2, seed=8)
