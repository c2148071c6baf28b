"""CPU oracle for the SDM coalescence hot path -- TEST INFRASTRUCTURE ONLY.

Thin ctypes access to ``oracle/sdm_oracle.c`` (plain C, fp64, single thread, written from the
paper).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package; the product (``paper_2101_06318_b200``)
never does, and this package imports nothing from the product.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build as _build

KERNEL_GOLOVIN = 0
KERNEL_GRAVITATIONAL = 1
KERNEL_GRAVITATIONAL_TABULATED = 2
KERNEL_USER = 3

_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        L = _lib
        p = C.c_void_p
        L.orc_philox4x32_10.argtypes = [p, p, p]
        L.orc_philox4x32_10.restype = None
        L.orc_rng.argtypes = [C.c_int64, p, C.c_uint64, C.c_uint64, p, p]
        L.orc_rng.restype = None
        L.orc_cell_start.argtypes = [C.c_int64, p, C.c_int32, p]
        L.orc_cell_start.restype = C.c_int
        L.orc_permutation.argtypes = [C.c_int64, p, p, p, p]
        L.orc_permutation.restype = None
        L.orc_cbrt_spec.argtypes = [C.c_double]
        L.orc_cbrt_spec.restype = C.c_double
        L.orc_kernel.argtypes = [C.c_int32, C.c_double, C.c_double, C.c_double]
        L.orc_kernel.restype = C.c_double
        L.orc_set_efficiency_table.argtypes = [C.c_int32, p, p]
        L.orc_set_efficiency_table.restype = C.c_int
        L.orc_efficiency.argtypes = [C.c_double, C.c_double]
        L.orc_efficiency.restype = C.c_double
        L.orc_set_user_kernel.argtypes = [p, p, C.c_int32]
        L.orc_set_user_kernel.restype = None
        L.orc_pair_probability.argtypes = [C.c_double, C.c_int64, C.c_int64, C.c_double, C.c_double]
        L.orc_pair_probability.restype = C.c_double
        L.orc_gamma_tilde.argtypes = [C.c_double, C.c_double, C.c_int64, C.c_int64]
        L.orc_gamma_tilde.restype = C.c_int64
        L.orc_collide_pair.argtypes = [p, p, p, p, C.c_int64]
        L.orc_collide_pair.restype = None
        L.orc_step.argtypes = [C.c_int64, p, p, p, C.c_int32, p, C.c_double, C.c_double, C.c_int32,
                               C.c_double, C.c_uint64, C.c_uint64, p, p, p]
        L.orc_step.restype = C.c_int
        L.orc_remove_zero.argtypes = [C.c_int64, p, p, p]
        L.orc_remove_zero.restype = C.c_int64
        L.orc_spectrum.argtypes = [C.c_int64, p, p, C.c_int32, p, p, C.c_double, C.c_double, C.c_int32, p]
        L.orc_spectrum.restype = None
        L.orc_collide_pair_attr.argtypes = [p, p, C.c_int32, C.c_int64, C.c_int64, C.c_int64, C.c_int64]
        L.orc_collide_pair_attr.restype = None
        L.orc_step_attr.argtypes = [C.c_int64, p, p, C.c_int32, C.c_int64, p, C.c_int32, p, C.c_double, C.c_double,
                                    C.c_int32, C.c_double, C.c_uint64, C.c_uint64, p, p, p]
        L.orc_step_attr.restype = C.c_int
        L.orc_remove_zero_attr.argtypes = [C.c_int64, p, p, C.c_int32, C.c_int64, p]
        L.orc_remove_zero_attr.restype = C.c_int64
        L.orc_moments.argtypes = [C.c_int64, p, p, p, C.c_int32, C.c_int32, p, p, p]
        L.orc_moments.restype = None
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _chk(a, dtype):
    assert isinstance(a, np.ndarray) and a.dtype == dtype and a.flags.c_contiguous, (a.dtype, dtype)
    return a


def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_ptr(c), _ptr(k), _ptr(out))
    return out


def rng(n, seed, step, sid=None):
    key64 = np.empty(n, dtype=np.uint64)
    ucand = np.empty(n, dtype=np.float64)
    if sid is not None:
        sid = _chk(np.ascontiguousarray(sid, dtype=np.int64), np.int64)
    lib().orc_rng(n, _ptr(sid), seed, step, _ptr(key64), _ptr(ucand))
    return key64, ucand


def cell_start(cell_id, n_cell) -> np.ndarray:
    cell_id = _chk(cell_id, np.int32)
    cs = np.empty(n_cell + 1, dtype=np.int32)
    rc = lib().orc_cell_start(cell_id.shape[0], _ptr(cell_id), n_cell, _ptr(cs))
    if rc != 0:
        raise ValueError("cell id out of range")
    return cs


def permutation(cell_id, key64, sid=None) -> np.ndarray:
    cell_id = _chk(cell_id, np.int32)
    key64 = _chk(key64, np.uint64)
    if sid is not None:
        sid = _chk(np.ascontiguousarray(sid, dtype=np.int64), np.int64)
    idx = np.empty(cell_id.shape[0], dtype=np.int32)
    lib().orc_permutation(cell_id.shape[0], _ptr(cell_id), _ptr(key64), _ptr(sid), _ptr(idx))
    return idx


def cbrt_spec(x: float) -> float:
    return lib().orc_cbrt_spec(float(x))


def kernel(ktype: int, kparam: float, vj: float, vk: float) -> float:
    return lib().orc_kernel(ktype, float(kparam), float(vj), float(vk))


def set_efficiency_table(r_grid, E):
    """Collection-efficiency table of KERNEL_GRAVITATIONAL_TABULATED: E[n_r, n_r] on the radius grid r_grid."""
    r_grid = _chk(np.ascontiguousarray(r_grid, dtype=np.float64), np.float64)
    E = _chk(np.ascontiguousarray(E, dtype=np.float64), np.float64)
    assert E.shape == (r_grid.shape[0], r_grid.shape[0])
    if lib().orc_set_efficiency_table(r_grid.shape[0], _ptr(r_grid), _ptr(E)) != 0:
        raise ValueError("invalid efficiency table")


_user_lib = None   # keeps the compiled user kernel alive


def set_user_kernel(c_source: str, params=()):
    """KERNEL_USER: compiles ``c_source`` -- plain C defining ``double sdm_user_kernel(double vj, double vk, const double
    *params)`` -- with gcc (-O2 -ffp-contract=off, like the oracle itself) and hands the function to the oracle as a
    callback.  Test infrastructure: the GPU library receives the same text as CUDA source (NVRTC, --fmad=false)."""
    import os
    import subprocess
    import tempfile

    global _user_lib
    d = tempfile.mkdtemp(prefix="orc_user_")
    src, so = os.path.join(d, "user_kernel.c"), os.path.join(d, "libuser_kernel.so")
    with open(src, "w") as f:
        f.write("#include <math.h>\n" + c_source + "\n")
    subprocess.run(["gcc", "-std=c11", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared", "-o", so, src,
                    "-lm"], check=True)
    _user_lib = C.CDLL(so)
    fn = C.cast(_user_lib.sdm_user_kernel, C.c_void_p)
    par = np.ascontiguousarray(np.asarray(params, dtype=np.float64))
    lib().orc_set_user_kernel(fn, _ptr(par) if par.size else None, int(par.size))


def efficiency(rj: float, rk: float) -> float:
    return lib().orc_efficiency(float(rj), float(rk))


def pair_probability(K: float, xi_max: int, n_s: int, dt: float, dV: float) -> float:
    return lib().orc_pair_probability(float(K), int(xi_max), int(n_s), float(dt), float(dV))


def gamma_tilde(p: float, u: float, xi_j: int, xi_k: int) -> int:
    return lib().orc_gamma_tilde(float(p), float(u), int(xi_j), int(xi_k))


def collide_pair(xi_a: int, v_a: float, xi_b: int, v_b: float, gamma: int):
    """Fig. 5 body for the pair (first, second) with uncapped gamma -> (xi_a, v_a, xi_b, v_b)."""
    xa, xb = C.c_int64(xi_a), C.c_int64(xi_b)
    va, vb = C.c_double(v_a), C.c_double(v_b)
    lib().orc_collide_pair(C.byref(xa), C.byref(va), C.byref(xb), C.byref(vb), int(gamma))
    return xa.value, va.value, xb.value, vb.value


def step(xi, v, cell_id, n_cell, dt, dV, ktype, kparam, seed, step, sid=None, want_perm=True):
    """One coalescence step IN PLACE on (xi, v).  Returns (idx, cell_start, n_events)."""
    xi = _chk(xi, np.int64)
    v = _chk(v, np.float64)
    cell_id = _chk(cell_id, np.int32)
    n = xi.shape[0]
    assert v.shape[0] == n and cell_id.shape[0] == n
    if sid is not None:
        sid = _chk(np.ascontiguousarray(sid, dtype=np.int64), np.int64)
    idx = np.empty(n, dtype=np.int32) if want_perm else None
    cs = np.empty(n_cell + 1, dtype=np.int32) if want_perm else None
    nev = C.c_int64(0)
    rc = lib().orc_step(n, _ptr(xi), _ptr(v), _ptr(cell_id), n_cell, _ptr(sid), float(dt), float(dV),
                        int(ktype), float(kparam), int(seed), int(step), _ptr(idx), _ptr(cs),
                        C.byref(nev))
    if rc != 0:
        raise ValueError("orc_step: invalid input")
    return idx, cs, nev.value


def collide_pair_attr(xi, attr, a, b, gamma):
    """Fig. 5 body IN PLACE on xi[n] and the row-major attribute block attr[n_attr, n] (row 0 = volume)
    for the pair (a = first-in-pair, b) with uncapped gamma."""
    xi = _chk(xi, np.int64)
    attr = _chk(attr, np.float64)
    assert attr.ndim == 2 and attr.shape[1] == xi.shape[0]
    lib().orc_collide_pair_attr(_ptr(xi), _ptr(attr), attr.shape[0], attr.shape[1], int(a), int(b), int(gamma))


def step_attr(xi, attr, cell_id, n_cell, dt, dV, ktype, kparam, seed, step, want_perm=True):
    """One coalescence step IN PLACE on xi[n] and attr[n_attr, n] (row 0 = volume).
    Returns (idx, cell_start, n_events)."""
    xi = _chk(xi, np.int64)
    attr = _chk(attr, np.float64)
    cell_id = _chk(cell_id, np.int32)
    n = xi.shape[0]
    assert attr.ndim == 2 and attr.shape[1] == n and cell_id.shape[0] == n
    idx = np.empty(n, dtype=np.int32) if want_perm else None
    cs = np.empty(n_cell + 1, dtype=np.int32) if want_perm else None
    nev = C.c_int64(0)
    rc = lib().orc_step_attr(n, _ptr(xi), _ptr(attr), attr.shape[0], n, _ptr(cell_id), n_cell, None, float(dt),
                             float(dV), int(ktype), float(kparam), int(seed), int(step), _ptr(idx), _ptr(cs),
                             C.byref(nev))
    if rc != 0:
        raise ValueError("orc_step_attr: invalid input")
    return idx, cs, nev.value


def remove_zero_attr(xi, attr, cell_id):
    """Stable removal of xi == 0 with all attribute rows.  Returns trimmed COPIES (xi, attr, cell_id)."""
    xi = _chk(xi, np.int64).copy()
    attr = _chk(attr, np.float64).copy()
    cell_id = _chk(cell_id, np.int32).copy()
    m = lib().orc_remove_zero_attr(xi.shape[0], _ptr(xi), _ptr(attr), attr.shape[0], attr.shape[1], _ptr(cell_id))
    return xi[:m].copy(), np.ascontiguousarray(attr[:, :m]), cell_id[:m].copy()


def remove_zero(xi, v, cell_id):
    """Stable removal of xi == 0.  Returns trimmed COPIES (xi, v, cell_id)."""
    xi = _chk(xi, np.int64).copy()
    v = _chk(v, np.float64).copy()
    cell_id = _chk(cell_id, np.int32).copy()
    m = lib().orc_remove_zero(xi.shape[0], _ptr(xi), _ptr(v), _ptr(cell_id))
    return xi[:m].copy(), v[:m].copy(), cell_id[:m].copy()


def moments(xi, v, cell_id=None, n_cell=1, per_cell=False):
    xi = _chk(xi, np.int64)
    v = _chk(v, np.float64)
    nout = n_cell if per_cell else 1
    if per_cell:
        cell_id = _chk(cell_id, np.int32)
    m0 = np.zeros(nout, dtype=np.int64)
    m1 = np.zeros(nout, dtype=np.float64)
    m2 = np.zeros(nout, dtype=np.float64)
    lib().orc_moments(xi.shape[0], _ptr(xi), _ptr(v), _ptr(cell_id) if per_cell else None,
                      n_cell, 1 if per_cell else 0, _ptr(m0), _ptr(m1), _ptr(m2))
    if per_cell:
        return m0, m1, m2
    return int(m0[0]), float(m1[0]), float(m2[0])


def spectrum(xi, v, v_edges, dlnr, rho, V, n_smooth=2):
    """Mass density per unit ln r on the bins v_edges (R17)."""
    xi = _chk(xi, np.int64)
    v = _chk(v, np.float64)
    v_edges = _chk(np.ascontiguousarray(v_edges, dtype=np.float64), np.float64)
    dlnr = _chk(np.ascontiguousarray(dlnr, dtype=np.float64), np.float64)
    nb = dlnr.shape[0]
    assert v_edges.shape[0] == nb + 1
    out = np.zeros(nb, dtype=np.float64)
    lib().orc_spectrum(xi.shape[0], _ptr(xi), _ptr(v), nb, _ptr(v_edges), _ptr(dlnr), float(rho), float(V),
                       int(n_smooth), _ptr(out))
    return out
