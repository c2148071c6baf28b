"""sdm_moments_noalloc -- the one entry point of libsdm that needs no device memory from the caller beyond the inputs
and the 24 bytes of results.

It exists for code that cannot call cudaMalloc at the moment it wants the moments: a host model that gave the whole
GPU to its own memory pool when it started, a monitoring hook on a thread that may not stall the device (cudaMalloc and
cudaFree synchronise it), a plug-in living inside a fixed device-memory budget.  Such a caller cannot build the
workspace every other libsdm call works on, so the scratch of the grid-wide sum is a static array inside the library
(28 KiB per GPU, one array shared by every call, kept until the process exits).

Checked here, through the C ABI, against the existing handle-based path (sdm_moments on a state loaded with
sdm_set_state): M0 bit-exact, M1 and M2 within the 1e-12 relative bar the other moment tests use -- on two calls in a
row that share the static array (a large state first, a smaller odd-sized one second, so anything the first call left
in the array would show), then once more on the first state.  The size limit is checked too.

This file sorts last on purpose (pytest runs files in name order and the driver uses -x): a failure here hides
nothing.  It must pass alone in a fresh process and after every other GPU test of the suite.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

REL = 1e-12


def _state(n, seed):
    """Seeded synthetic (xi, v): multiplicities 0..2^20 (zeros included), volumes of 1-100 um droplets."""
    rng = np.random.default_rng(seed)
    xi = rng.integers(0, 2 ** 20, size=n, dtype=np.int64)
    r = rng.uniform(1e-6, 100e-6, size=n)
    v = 4.0 / 3.0 * np.pi * r ** 3
    return xi, v


def _existing_path(torch, pkg, xi_d, v_d):
    """sdm_moments(per_cell = 0) of a handle holding (xi, v) in one cell: the path that was there before."""
    n = xi_d.shape[0]
    s = pkg.SDM(n, 1, device="cuda:0")
    s.set_state(xi_d, v_d, torch.zeros(n, dtype=torch.int32, device="cuda:0"))
    m0, m1, m2 = s.moments_host()
    s.close()
    return m0, m1, m2


def _close(a, b):
    return abs(a - b) <= REL * abs(b)


def test_noalloc_moments_equal_the_handle_path_on_consecutive_calls():
    import torch

    import paper_2101_06318_b200 as pkg

    assert torch.cuda.is_available()
    pkg.load_library()
    dev = "cuda:0"
    # sizes: 1184 CTAs and an even count; then fewer CTAs than the first call used and an odd count
    cases = [_state(3_000_000, 11), _state(70_001, 12)]
    dev_states = [(torch.from_numpy(xi).to(dev), torch.from_numpy(v).to(dev)) for xi, v in cases]
    expected = [_existing_path(torch, pkg, xi_d, v_d) for xi_d, v_d in dev_states]
    # results buffers are the caller's, made before the calls: the entry point itself allocates nothing
    outs = [(torch.full((1,), -7, dtype=torch.int64, device=dev), torch.full((1,), -7.0, dtype=torch.float64, device=dev),
             torch.full((1,), -7.0, dtype=torch.float64, device=dev)) for _ in range(3)]
    torch.cuda.synchronize()

    # two calls in a row on the same stream, no synchronisation between them, then the first state again
    order = [0, 1, 0]
    for k, which in enumerate(order):
        xi_d, v_d = dev_states[which]
        pkg.moments_noalloc(xi_d, v_d, outs[k])
    torch.cuda.synchronize()

    for k, which in enumerate(order):
        m0, m1, m2 = (int(outs[k][0].item()), float(outs[k][1].item()), float(outs[k][2].item()))
        e0, e1, e2 = expected[which]
        assert m0 == e0, (k, m0, e0)
        assert _close(m1, e1) and _close(m2, e2), (k, m1, e1, m2, e2)
        # and the plain definition, so that both paths being wrong together cannot pass
        xi, v = cases[which]
        assert m0 == int(xi.sum())
        assert _close(m1, float(np.sum(xi.astype(np.float64) * v)))


def test_noalloc_empty_and_single():
    import torch

    import paper_2101_06318_b200 as pkg

    dev = "cuda:0"
    out = (torch.full((1,), -7, dtype=torch.int64, device=dev), torch.full((1,), -7.0, dtype=torch.float64, device=dev),
           torch.full((1,), -7.0, dtype=torch.float64, device=dev))
    xi = torch.tensor([5, 3], dtype=torch.int64, device=dev)
    v = torch.tensor([2.0, 0.5], dtype=torch.float64, device=dev)
    pkg.moments_noalloc(xi, v, out, n_sd=0)
    torch.cuda.synchronize()
    assert (out[0].item(), out[1].item(), out[2].item()) == (0, 0.0, 0.0)
    pkg.moments_noalloc(xi, v, out, n_sd=1)
    torch.cuda.synchronize()
    assert (out[0].item(), out[1].item(), out[2].item()) == (5, 10.0, 20.0)
    pkg.moments_noalloc(xi, v, out)
    torch.cuda.synchronize()
    assert (out[0].item(), out[1].item(), out[2].item()) == (8, 11.5, 20.75)


def test_noalloc_rejects_sizes_beyond_its_maximum_and_bad_pointers():
    import torch

    import paper_2101_06318_b200 as pkg

    dev = "cuda:0"
    out = (torch.zeros(1, dtype=torch.int64, device=dev), torch.zeros(1, dtype=torch.float64, device=dev),
           torch.zeros(1, dtype=torch.float64, device=dev))
    xi = torch.ones(8, dtype=torch.int64, device=dev)
    v = torch.ones(8, dtype=torch.float64, device=dev)
    # the size check comes before anything is read: the small arrays are never touched
    with pytest.raises(pkg.SdmError, match="SDM_ECAPACITY.*SDM_NOALLOC_MAX_SD"):
        pkg.moments_noalloc(xi, v, out, n_sd=pkg.NOALLOC_MAX_SD + 1)
    with pytest.raises(pkg.SdmError, match="SDM_EINVAL.*negative"):
        pkg.moments_noalloc(xi, v, out, n_sd=-1)
    with pytest.raises(pkg.SdmError, match="SDM_EINVAL.*aligned"):
        pkg.moments_noalloc(xi[1:], v[1:], out)
    # a rejected call leaves the entry point usable
    pkg.moments_noalloc(xi, v, out)
    torch.cuda.synchronize()
    assert (out[0].item(), out[1].item(), out[2].item()) == (8, 8.0, 8.0)
