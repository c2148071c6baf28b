"""ctypes binding of include/sdm.h -- argument marshalling only.

Every step of the hot path runs inside libsdm.so's CUDA kernels.  Names mirror the C ABI:
``SDM.set_state`` -> ``sdm_set_state``, ``SDM.coalescence_step`` -> ``sdm_coalescence_step``, ...
"""
from __future__ import annotations

import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))

KERNEL_GOLOVIN = 0
KERNEL_GRAVITATIONAL = 1
KERNEL_GRAVITATIONAL_TABULATED = 2
KERNEL_USER = 3
OPT_FORCE_GENERAL = 1
OPT_SEGMENT_CAP = 2
OPT_WRITE_IDX = 3
OPT_SCREENING = 4
OPT_TIMING = 5
OPT_LANES_PER_CELL = 6
OPT_SORT_ENGINE = 7
OPT_DETERMINISTIC = 8
OPT_CTAS_PER_SM = 9
OPT_BOX_CTAS = 10
OPT_BOX_REGION_CAP = 11
OPT_BOX_SORT_CAP = 12
OPT_COOPERATIVE = 13
CNT_NAMES = ("n_sd", "events", "zeros", "launches", "mode", "max_cell", "exact_evals", "reserved")

SDM_OK, SDM_EINVAL, SDM_ECAPACITY, SDM_ECUDA, SDM_ESTATE = 0, -1, -2, -3, -4
_CODES = {-1: "SDM_EINVAL", -2: "SDM_ECAPACITY", -3: "SDM_ECUDA", -4: "SDM_ESTATE"}

# every symbol include/sdm.h declares (tests check the header against this and the .so)
SYMBOLS = (
    "sdm_version", "sdm_workspace_bytes", "sdm_create", "sdm_destroy", "sdm_set_option",
    "sdm_set_state", "sdm_set_state_host", "sdm_get_state", "sdm_get_state_host",
    "sdm_coalescence_step", "sdm_coalescence_step_moments", "sdm_remove_zero", "sdm_moments", "sdm_moments_host",
    "sdm_get_permutation", "sdm_run", "sdm_get_counters", "sdm_get_timing", "sdm_last_error",
    "sdm_workspace_bytes_attr", "sdm_create_attr", "sdm_set_attributes", "sdm_get_attributes",
    "sdm_set_efficiency_table", "sdm_spectrum", "sdm_set_cell_id", "sdm_set_index_base", "sdm_set_kernel_source", "sdm_debug_permutation",
    "sdm_moments_noalloc",
)
MAX_ATTR = 8


class SdmError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{_CODES.get(code, code)}: {msg}")
        self.code = code


class KernelDesc(C.Structure):
    _fields_ = [("type", C.c_int32), ("reserved", C.c_int32), ("b", C.c_double), ("E", C.c_double)]


_lib = None


def library_path() -> str:
    """In-tree libsdm.so; SDM_LIBRARY overrides the path (to try an alternative build of the same ABI)."""
    return os.environ.get("SDM_LIBRARY") or os.path.join(HERE, "libsdm.so")


def load_library() -> C.CDLL:
    """Loads the in-tree libsdm.so.  Raises (never falls back) if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    path = library_path()
    if not os.path.exists(path):
        raise ImportError(f"{path} is missing: run `python -m paper_2101_06318_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(path)
    vp, i64, i32, u64, dbl = C.c_void_p, C.c_int64, C.c_int32, C.c_uint64, C.c_double
    L.sdm_version.restype = C.c_int
    L.sdm_workspace_bytes.argtypes = [i64, i32]
    L.sdm_workspace_bytes.restype = C.c_size_t
    L.sdm_create.argtypes = [C.POINTER(vp), i64, i32, vp, C.c_size_t, vp]
    L.sdm_workspace_bytes_attr.argtypes = [i64, i32, i32]
    L.sdm_workspace_bytes_attr.restype = C.c_size_t
    L.sdm_create_attr.argtypes = [C.POINTER(vp), i64, i32, i32, vp, C.c_size_t, vp]
    L.sdm_set_attributes.argtypes = [vp, vp, i64]
    L.sdm_get_attributes.argtypes = [vp, vp, i64]
    L.sdm_set_efficiency_table.argtypes = [vp, i32, vp, vp]
    L.sdm_set_cell_id.argtypes = [vp, vp]
    L.sdm_set_index_base.argtypes = [vp, i64]
    L.sdm_debug_permutation.argtypes = [vp, vp]
    L.sdm_set_kernel_source.argtypes = [vp, C.c_char_p, i32, vp]
    L.sdm_spectrum.argtypes = [vp, i32, vp, vp, dbl, dbl, i32, vp]
    L.sdm_destroy.argtypes = [vp]
    L.sdm_set_option.argtypes = [vp, i32, i64]
    L.sdm_set_state.argtypes = [vp, i64, vp, vp, vp]
    L.sdm_set_state_host.argtypes = [vp, i64, vp, vp, vp]
    L.sdm_get_state.argtypes = [vp, C.POINTER(i64), vp, vp, vp]
    L.sdm_get_state_host.argtypes = [vp, C.POINTER(i64), vp, vp, vp]
    L.sdm_coalescence_step.argtypes = [vp, dbl, dbl, C.POINTER(KernelDesc), u64, u64]
    L.sdm_coalescence_step_moments.argtypes = [vp, dbl, dbl, C.POINTER(KernelDesc), u64, u64, vp, vp, vp]
    L.sdm_remove_zero.argtypes = [vp, C.POINTER(i64)]
    L.sdm_moments.argtypes = [vp, C.c_int, vp, vp, vp]
    L.sdm_moments_host.argtypes = [vp, C.c_int, vp, vp, vp]
    L.sdm_get_permutation.argtypes = [vp, vp, vp]
    L.sdm_run.argtypes = [vp, dbl, dbl, C.POINTER(KernelDesc), u64, u64, i64, C.c_int]
    L.sdm_get_counters.argtypes = [vp, C.POINTER(i64)]
    L.sdm_get_timing.argtypes = [vp, C.POINTER(dbl), C.POINTER(i64)]
    L.sdm_moments_noalloc.argtypes = [vp, vp, i64, vp, vp, vp, vp, C.c_char_p, C.c_size_t]
    L.sdm_last_error.argtypes = [vp]
    L.sdm_last_error.restype = C.c_char_p
    for name in SYMBOLS:
        if name not in ("sdm_workspace_bytes", "sdm_workspace_bytes_attr", "sdm_last_error"):
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


def version() -> int:
    return load_library().sdm_version()


def workspace_bytes(capacity: int, n_cell: int, n_attr: int = 1) -> int:
    return int(load_library().sdm_workspace_bytes_attr(capacity, n_cell, n_attr))


NOALLOC_MAX_SD = 2139095040


def moments_noalloc(xi, v, out, stream=None, n_sd=None):
    """sdm_moments_noalloc: global moments of (xi, v) without a handle or a workspace, for code that cannot allocate
    device memory when it needs them (everything on the device already belongs to someone's pool, or the thread must
    not stall the device in cudaMalloc).  The reduction's scratch is a static 28 KiB array inside libsdm, one per GPU,
    shared by every call: calls that may overlap on the GPU race, so keep them ordered (one stream).  Nothing is
    allocated here either: `out` = (m0 int64[1], m1 float64[1], m2 float64[1]) device tensors supplied by the caller,
    written asynchronously on `stream` (default: torch's current stream of xi's device).  n_sd defaults to len(xi).
    The first call on a device should come before any stream capture."""
    import torch

    lib = load_library()
    n = int(xi.shape[0] if n_sd is None else n_sd)
    assert xi.is_cuda and v.is_cuda and xi.dtype == torch.int64 and v.dtype == torch.float64
    assert xi.is_contiguous() and v.is_contiguous()
    m0, m1, m2 = out
    assert m0.is_cuda and m0.dtype == torch.int64 and m1.dtype == torch.float64 and m2.dtype == torch.float64
    err = C.create_string_buffer(256)
    with torch.cuda.device(xi.device):
        s = stream if stream is not None else torch.cuda.current_stream(xi.device)
        rc = lib.sdm_moments_noalloc(C.c_void_p(xi.data_ptr()), C.c_void_p(v.data_ptr()), n, C.c_void_p(m0.data_ptr()),
                                     C.c_void_p(m1.data_ptr()), C.c_void_p(m2.data_ptr()), C.c_void_p(s.cuda_stream),
                                     err, len(err))
    if rc != SDM_OK:
        raise SdmError(rc, err.value.decode())
    return out


def _kernel(kernel: int, kparam: float) -> KernelDesc:
    if kernel == KERNEL_GOLOVIN:
        return KernelDesc(KERNEL_GOLOVIN, 0, float(kparam), 0.0)
    return KernelDesc(int(kernel), 0, 0.0, float(kparam))


class SDM:
    """One simulation state on one GPU.  Device memory (workspace) is a torch tensor; the stream is
    torch's current stream at construction."""

    def __init__(self, capacity: int, n_cell: int, device="cuda:0", stream=None, n_attr: int = 1):
        import torch

        self._lib = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: libsdm has no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        self.capacity, self.n_cell, self.n_attr = int(capacity), int(n_cell), int(n_attr)
        nbytes = workspace_bytes(self.capacity, self.n_cell, self.n_attr)
        if nbytes == 0:
            raise SdmError(SDM_EINVAL, "invalid capacity / n_cell / n_attr")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = self.workspace.data_ptr()
            self._ws_ptr = (base + 255) // 256 * 256
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            h = C.c_void_p()
            rc = self._lib.sdm_create_attr(C.byref(h), self.capacity, self.n_cell, self.n_attr,
                                           C.c_void_p(self._ws_ptr), nbytes, C.c_void_p(self.stream.cuda_stream))
        if rc != SDM_OK:
            raise SdmError(rc, self._lib.sdm_last_error(None).decode())
        self._h = h

    # -- helpers ------------------------------------------------------------------------------
    def _check(self, rc: int):
        if rc != SDM_OK:
            raise SdmError(rc, self._lib.sdm_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            self._lib.sdm_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @staticmethod
    def _p(t):
        return None if t is None else C.c_void_p(t.data_ptr())

    def _dev(self, t, dtype):
        assert t.is_cuda and t.dtype == dtype and t.is_contiguous(), (t.device, t.dtype)
        return t

    def _host(self, t, dtype):
        assert (not t.is_cuda) and t.dtype == dtype and t.is_contiguous(), (t.device, t.dtype)
        return t

    # -- the C ABI, one method per entry point ---------------------------------------------------
    def set_option(self, option: int, value: int):
        self._check(self._lib.sdm_set_option(self._h, option, int(value)))

    def set_state(self, xi, v, cell_id):
        """xi int64, v float64, cell_id int32 torch tensors on the device."""
        t = self.torch
        n = xi.shape[0]
        self._dev(xi, t.int64), self._dev(v, t.float64), self._dev(cell_id, t.int32)
        self._check(self._lib.sdm_set_state(self._h, n, self._p(xi), self._p(v), self._p(cell_id)))

    def set_state_host(self, xi, v, cell_id):
        """Same, from host tensors (pinned recommended): the H2D copies are part of the call."""
        t = self.torch
        n = xi.shape[0]
        self._host(xi, t.int64), self._host(v, t.float64), self._host(cell_id, t.int32)
        self._check(self._lib.sdm_set_state_host(self._h, n, self._p(xi), self._p(v), self._p(cell_id)))

    def spectrum(self, v_edges, dlnr, rho, V, n_smooth=2):
        """Mass density per unit ln r on the bins v_edges (numpy float64 host arrays in, numpy array out)."""
        import numpy as np

        v_edges = np.ascontiguousarray(v_edges, dtype=np.float64)
        dlnr = np.ascontiguousarray(dlnr, dtype=np.float64)
        assert v_edges.shape[0] == dlnr.shape[0] + 1
        out = np.zeros(dlnr.shape[0], dtype=np.float64)
        self._check(self._lib.sdm_spectrum(self._h, int(dlnr.shape[0]), v_edges.ctypes.data_as(C.c_void_p),
                                           dlnr.ctypes.data_as(C.c_void_p), float(rho), float(V), int(n_smooth),
                                           out.ctypes.data_as(C.c_void_p)))
        return out

    def set_efficiency_table(self, r_grid, E):
        """Collection efficiencies for KERNEL_GRAVITATIONAL_TABULATED: numpy float64 r_grid[n_r], E[n_r, n_r]."""
        import numpy as np

        r_grid = np.ascontiguousarray(r_grid, dtype=np.float64)
        E = np.ascontiguousarray(E, dtype=np.float64)
        assert E.shape == (r_grid.shape[0], r_grid.shape[0])
        self._check(self._lib.sdm_set_efficiency_table(self._h, int(r_grid.shape[0]), r_grid.ctypes.data_as(C.c_void_p),
                                                       E.ctypes.data_as(C.c_void_p)))

    def set_cell_id(self, cell_id):
        """New cell ids (int32 device tensor, storage order, current n_sd entries) after displacement."""
        self._dev(cell_id, self.torch.int32)
        self._check(self._lib.sdm_set_cell_id(self._h, self._p(cell_id)))

    def set_kernel_source(self, cuda_src: str, params=()):
        """CUDA source defining ``__device__ double sdm_user_kernel(double vj, double vk, const double *params)`` for
        KERNEL_USER, compiled at run time (NVRTC); params: up to 16 floats."""
        import numpy as np

        par = np.ascontiguousarray(np.asarray(params, dtype=np.float64))
        self._check(self._lib.sdm_set_kernel_source(self._h, cuda_src.encode(), int(par.size),
                                                    par.ctypes.data_as(C.c_void_p) if par.size else None))

    def debug_permutation(self, keys):
        """Rows a2-a3 with caller-supplied sort keys (uint64 as an int64 device tensor, by storage index): the tie rule."""
        self._dev(keys, self.torch.int64)
        self._check(self._lib.sdm_debug_permutation(self._h, self._p(keys)))

    def set_index_base(self, base: int):
        """Global storage index of this handle's droplet 0 (sharded runs; see sdm_set_index_base)."""
        self._check(self._lib.sdm_set_index_base(self._h, int(base)))

    def set_attributes(self, attr):
        """Rows 1..n_attr-1 of the attribute block: a contiguous float64 device tensor [n_attr-1, n_sd]."""
        self._dev(attr, self.torch.float64)
        assert attr.dim() == 2 and attr.shape[0] == self.n_attr - 1
        self._check(self._lib.sdm_set_attributes(self._h, self._p(attr), int(attr.shape[1])))

    def get_attributes(self):
        """Returns rows 1..n_attr-1 as a device tensor [n_attr-1, n_sd] (current n_sd)."""
        t = self.torch
        n = self.counters()["n_sd"]
        out = t.empty((self.n_attr - 1, max(n, 1)), dtype=t.float64, device=self.device)
        self._check(self._lib.sdm_get_attributes(self._h, self._p(out), int(out.shape[1])))
        return out[:, :n]

    def get_state(self):
        """Returns (xi, v, cell_id) device tensors trimmed to the current n_sd."""
        t = self.torch
        xi = t.empty(self.capacity, dtype=t.int64, device=self.device)
        v = t.empty(self.capacity, dtype=t.float64, device=self.device)
        c = t.empty(self.capacity, dtype=t.int32, device=self.device)
        n = C.c_int64(0)
        self._check(self._lib.sdm_get_state(self._h, C.byref(n), self._p(xi), self._p(v), self._p(c)))
        return xi[: n.value], v[: n.value], c[: n.value]

    def get_state_host(self, xi, v, cell_id) -> int:
        """Copies the state into the given host tensors (capacity-sized); returns n_sd."""
        n = C.c_int64(0)
        self._check(self._lib.sdm_get_state_host(self._h, C.byref(n), self._p(xi), self._p(v), self._p(cell_id)))
        return n.value

    def coalescence_step(self, dt, dV, kernel, kparam, seed, step):
        k = _kernel(kernel, kparam)
        self._check(self._lib.sdm_coalescence_step(self._h, float(dt), float(dV), C.byref(k), int(seed), int(step)))

    def coalescence_step_moments(self, dt, dV, kernel, kparam, seed, step, out=None):
        """One step plus the global moments of the post-step state (device tensors, asynchronous)."""
        t = self.torch
        k = _kernel(kernel, kparam)
        if out is None:
            out = (t.empty(1, dtype=t.int64, device=self.device), t.empty(1, dtype=t.float64, device=self.device),
                   t.empty(1, dtype=t.float64, device=self.device))
        self._check(self._lib.sdm_coalescence_step_moments(self._h, float(dt), float(dV), C.byref(k), int(seed),
                                                           int(step), self._p(out[0]), self._p(out[1]), self._p(out[2])))
        return out

    def remove_zero(self, sync: bool = True):
        if not sync:
            self._check(self._lib.sdm_remove_zero(self._h, None))
            return None
        n = C.c_int64(0)
        self._check(self._lib.sdm_remove_zero(self._h, C.byref(n)))
        return n.value

    def moments(self, per_cell: bool = False, out=None):
        """Device-side moments (asynchronous): returns (m0 int64, m1, m2 float64) device tensors."""
        t = self.torch
        k = self.n_cell if per_cell else 1
        if out is None:
            out = (t.empty(k, dtype=t.int64, device=self.device), t.empty(k, dtype=t.float64, device=self.device),
                   t.empty(k, dtype=t.float64, device=self.device))
        self._check(self._lib.sdm_moments(self._h, 1 if per_cell else 0, self._p(out[0]), self._p(out[1]), self._p(out[2])))
        return out

    def moments_host(self, per_cell: bool = False):
        import numpy as np

        k = self.n_cell if per_cell else 1
        m0 = np.zeros(k, dtype=np.int64)
        m1 = np.zeros(k, dtype=np.float64)
        m2 = np.zeros(k, dtype=np.float64)
        self._check(self._lib.sdm_moments_host(self._h, 1 if per_cell else 0, m0.ctypes.data_as(C.c_void_p),
                                               m1.ctypes.data_as(C.c_void_p), m2.ctypes.data_as(C.c_void_p)))
        if per_cell:
            return m0, m1, m2
        return int(m0[0]), float(m1[0]), float(m2[0])

    def get_permutation(self, n_sd: int):
        """(idx[n_sd], cell_start[n_cell+1]) device tensors of the last coalescence step."""
        t = self.torch
        idx = t.empty(max(int(n_sd), 1), dtype=t.int32, device=self.device)
        cs = t.empty(self.n_cell + 1, dtype=t.int32, device=self.device)
        self._check(self._lib.sdm_get_permutation(self._h, self._p(idx), self._p(cs)))
        return idx[: int(n_sd)], cs

    def run(self, dt, dV, kernel, kparam, seed, step0, n_steps, remove_zero_each_step=True):
        k = _kernel(kernel, kparam)
        self._check(self._lib.sdm_run(self._h, float(dt), float(dV), C.byref(k), int(seed), int(step0),
                                      int(n_steps), 1 if remove_zero_each_step else 0))

    def timing(self):
        """(total_ms, n_launches) of the dominant kernel since the last call (needs OPT_TIMING)."""
        ms, cnt = C.c_double(0.0), C.c_int64(0)
        self._check(self._lib.sdm_get_timing(self._h, C.byref(ms), C.byref(cnt)))
        return ms.value, cnt.value

    def counters(self) -> dict:
        arr = (C.c_int64 * 8)()
        self._check(self._lib.sdm_get_counters(self._h, arr))
        return dict(zip(CNT_NAMES, [int(x) for x in arr]))
