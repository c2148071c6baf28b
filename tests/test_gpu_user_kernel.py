"""NEXT-2: user-supplied kernel code on the device (sdm_set_kernel_source, NVRTC) against the oracle running the SAME
source text as a C callback (gcc -ffp-contract=off): bit-exact on every path, with attributes, and a built-in kernel
re-expressed as user code reproduces the built-in step bit for bit."""
import numpy as np
import pytest

import oracle
import workloads

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

PRODUCT = "double sdm_user_kernel(double vj, double vk, const double *p) { return p[0] * vj * vk; }"
GOLOVIN = "double sdm_user_kernel(double vj, double vk, const double *p) { double s = vj + vk; return p[0] * s; }"
# a kernel that is neither symmetric nor smooth: exercises the (vj, vk) ordering and libm-free control flow
ASYM = ("double sdm_user_kernel(double vj, double vk, const double *p) "
        "{ double d = vj - vk; if (d < 0.0) d = -d; return p[0] * vj + p[1] * d * vk; }")


@pytest.fixture(scope="module")
def sdm_mod():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2101_06318_b200 as m
    m.load_library()
    return m


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _run(sdm_mod, w, c_src, params, steps, options=(), expect_mode=None, fused_moments=False):
    oracle.set_user_kernel(c_src, params)
    s = sdm_mod.SDM(w.n_sd, w.n_cell)
    for k, val in options:
        s.set_option(k, val)
    s.set_kernel_source("__device__ " + c_src, params)
    s.set_state(_dev(w.xi), _dev(w.v), _dev(w.cell_id))
    if expect_mode is not None:
        assert s.counters()["mode"] == expect_mode
    xi, v, cell = w.xi.copy(), w.v.copy(), w.cell_id.copy()
    events = 0
    for step in range(steps):
        xi, v, cell = oracle.remove_zero(xi, v, cell)
        assert s.remove_zero() == len(xi)
        idx, cs, nev = oracle.step(xi, v, cell, w.n_cell, w.dt, w.dV, oracle.KERNEL_USER, 0.0, w.seed, step)
        events += nev
        if fused_moments and step % 2:
            m = s.coalescence_step_moments(w.dt, w.dV, sdm_mod.KERNEL_USER, 0.0, w.seed, step)
            o = oracle.moments(xi, v)
            assert int(m[0].cpu()[0]) == o[0] and abs(float(m[1].cpu()[0]) - o[1]) <= 1e-12 * o[1]
        else:
            s.coalescence_step(w.dt, w.dV, sdm_mod.KERNEL_USER, 0.0, w.seed, step)
        gxi, gv, _ = (t.cpu().numpy() for t in s.get_state())
        gidx, gcs = (t.cpu().numpy() for t in s.get_permutation(len(xi)))
        assert np.array_equal(gidx, idx) and np.array_equal(gcs, cs), f"permutation differs at step {step}"
        assert np.array_equal(gxi, xi), f"xi differs at step {step}"
        assert np.array_equal(gv, v), f"v differs at step {step}"
    cnt = s.counters()
    assert cnt["events"] == events
    s.close()
    return events, len(xi)


def test_product_kernel_on_the_fused_general_and_box_paths(sdm_mod):
    w = workloads.grid_small_multiplicity(24, 24, 32, seed=2)             # v = 1, xi in 1..3
    events, n_end = _run(sdm_mod, w, PRODUCT, [0.02], 10, expect_mode=1, fused_moments=True)
    assert events > 3000 and n_end < w.n_sd
    w = workloads.grid_small_multiplicity(24, 24, 32, seed=3, shuffled=True)
    events, _ = _run(sdm_mod, w, PRODUCT, [0.02], 8, expect_mode=0)
    assert events > 3000
    n = 6000
    rng = np.random.default_rng(5)
    w = workloads.Workload("box", rng.integers(1, 4, n).astype(np.int64), rng.uniform(0.5, 2.0, n),
                           np.zeros(n, dtype=np.int32), 1, 1.0, 1.0, 0, 0.0, 0, seed=4)
    events, n_end = _run(sdm_mod, w, ASYM, [1e-4, 3e-5], 8, expect_mode=2)
    assert events > 1000 and n_end < n


def test_full_cells_counting_sort_kernel_and_an_asymmetric_kernel(sdm_mod):
    w = workloads.grid_uniform(10, 10, 256, seed=7)
    w.dV = 1.0
    rng = np.random.default_rng(1)
    w.xi[:] = rng.integers(1, 1000, w.n_sd)
    events, _ = _run(sdm_mod, w, ASYM, [2e8, 1e22], 6, expect_mode=1)
    assert events > 200


# R20: a kernel whose value is negative for some pairs, NaN for others (0/0) and a real collision rate for the rest
BAD_VALUES = ("double sdm_user_kernel(double vj, double vk, const double *p) "
              "{ double r = vj / vk; if (r > 1.5) return -p[0] * vj; if (r < 0.7) { double z = vj - vj; return z / z; } "
              "return p[0] * (vj + vk); }")


def test_negative_and_nan_kernel_values_are_no_event_on_every_path(sdm_mod):
    """DESIGN.md R20.  Volumes spread over 0.5..2 so that all three branches of BAD_VALUES are taken by many pairs;
    multiplicities never grow, events still happen, and device == oracle on the fused, general and box paths."""
    rng = np.random.default_rng(8)
    for shuffled, mode in ((False, 1), (True, 0)):
        w = workloads.grid_small_multiplicity(16, 16, 32, seed=12, shuffled=shuffled)
        w.v[:] = rng.uniform(0.5, 2.0, w.n_sd)
        events, n_end = _run(sdm_mod, w, BAD_VALUES, [0.02], 8, expect_mode=mode)
        assert events > 500 and n_end < w.n_sd
    n = 5000
    w = workloads.Workload("box", rng.integers(1, 4, n).astype(np.int64), rng.uniform(0.5, 2.0, n),
                           np.zeros(n, dtype=np.int32), 1, 1.0, 1.0, 0, 0.0, 0, seed=4)
    events, _ = _run(sdm_mod, w, BAD_VALUES, [2e-4], 6, expect_mode=2)
    assert events > 300
    # the three branches really occur among candidate pairs of such a state
    r = w.v[0::2] / w.v[1::2]
    assert (r > 1.5).sum() > 100 and (r < 0.7).sum() > 100 and ((r >= 0.7) & (r <= 1.5)).sum() > 100


def test_permutation_pass_of_a_user_kernel_step_does_not_count_exact_evaluations(sdm_mod):
    """With SDM_OPT_SCREENING = 0 the permutation pass in front of the user pair kernel (dt/dV = 0) used to evaluate and
    count every pair a second time.  Now each candidate pair is counted once per step (give or take the 2^-31 chance
    per droplet that its uniform word is 0 or 1)."""
    w = workloads.grid_uniform(6, 6, 256, seed=3)
    w.dV = 1.0
    oracle.set_user_kernel(PRODUCT, [1e-30])
    s = sdm_mod.SDM(w.n_sd, w.n_cell)
    s.set_option(sdm_mod.OPT_SCREENING, 0)
    s.set_kernel_source("__device__ " + PRODUCT, [1e-30])
    s.set_state(_dev(w.xi), _dev(w.v), _dev(w.cell_id))
    assert s.counters()["mode"] == 1
    for step in range(3):
        s.coalescence_step(w.dt, w.dV, sdm_mod.KERNEL_USER, 0.0, w.seed, step)
    assert s.counters()["exact_evals"] == 3 * (w.n_sd // 2)
    s.close()


def test_golovin_as_user_code_reproduces_the_builtin_kernel_bit_for_bit(sdm_mod):
    w = workloads.grid_poisson(24, 24, 64.0, shuffled=False, seed=6)
    w.kparam = 1500.0 * 4000.0
    a = sdm_mod.SDM(w.n_sd, w.n_cell)
    b = sdm_mod.SDM(w.n_sd, w.n_cell)
    b.set_kernel_source("__device__ " + GOLOVIN, [w.kparam])
    for s in (a, b):
        s.set_state(_dev(w.xi), _dev(w.v), _dev(w.cell_id))
    for step in range(10):
        a.coalescence_step(w.dt, w.dV, sdm_mod.KERNEL_GOLOVIN, w.kparam, 9, step)
        b.coalescence_step(w.dt, w.dV, sdm_mod.KERNEL_USER, 0.0, 9, step)
    for ta, tb in zip(a.get_state(), b.get_state()):
        assert torch.equal(ta, tb)
    assert a.counters()["events"] == b.counters()["events"] > 100
    assert torch.equal(a.get_permutation(w.n_sd)[0], b.get_permutation(w.n_sd)[0])
    a.close(), b.close()


def test_user_kernel_updates_every_attribute_row(sdm_mod):
    w = workloads.grid_small_multiplicity(12, 12, 32, seed=11)
    rng = np.random.default_rng(3)
    extra = rng.integers(0, 50, (2, w.n_sd)).astype(np.float64)
    oracle.set_user_kernel(PRODUCT, [0.03])
    s = sdm_mod.SDM(w.n_sd, w.n_cell, n_attr=3)
    s.set_kernel_source("__device__ " + PRODUCT, [0.03])
    s.set_state(_dev(w.xi), _dev(w.v), _dev(w.cell_id))
    s.set_attributes(_dev(extra))
    xi = w.xi.copy()
    attr = np.ascontiguousarray(np.vstack([w.v[None, :], extra]))
    for step in range(5):
        oracle.step_attr(xi, attr, w.cell_id, w.n_cell, w.dt, w.dV, oracle.KERNEL_USER, 0.0, w.seed, step)
        s.coalescence_step(w.dt, w.dV, sdm_mod.KERNEL_USER, 0.0, w.seed, step)
    gxi, gv, _ = (t.cpu().numpy() for t in s.get_state())
    assert np.array_equal(gxi, xi) and np.array_equal(gv, attr[0])
    assert np.array_equal(s.get_attributes().cpu().numpy(), attr[1:])
    s.close()


def test_errors_compile_log_missing_source_and_too_many_parameters(sdm_mod):
    s = sdm_mod.SDM(64, 2)
    s.set_state(_dev(np.ones(4, dtype=np.int64)), _dev(np.ones(4)), _dev(np.zeros(4, dtype=np.int32)))
    with pytest.raises(sdm_mod.SdmError) as e:                      # SDM_KERNEL_USER before any source
        s.coalescence_step(1.0, 1.0, sdm_mod.KERNEL_USER, 0.0, 0, 0)
    assert e.value.code == -1
    with pytest.raises(sdm_mod.SdmError) as e:
        s.set_kernel_source("__device__ double sdm_user_kernel(double vj, double vk, const double *p) { return undefined_name; }")
    assert e.value.code == -1 and "undefined_name" in str(e.value)
    with pytest.raises(sdm_mod.SdmError):
        s.set_kernel_source("__device__ " + PRODUCT, list(range(17)))
    s.set_kernel_source("__device__ " + PRODUCT, [1.0])             # a good source after a bad one
    s.coalescence_step(1.0, 1.0, sdm_mod.KERNEL_USER, 0.0, 0, 0)
    s.close()
