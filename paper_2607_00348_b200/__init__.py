"""paper_2607_00348_b200 -- B200-native Transit Least Squares period search (GTLS hot path).

Thin Python binding over ``libgtls.so`` (C ABI in ``include/gtls.h``): argument marshalling
only -- every step of the search runs in the library's CUDA kernels.  The functions keep the
names of the C entry points.  Arrays may be

* ``torch`` CUDA tensors (float64): passed as device pointers; outputs are CUDA tensors and the
  work is enqueued on torch's current stream (or ``stream=``);
* ``numpy`` arrays: passed as host pointers; the library copies to / from the device itself.

PyTorch is used for device memory and streams only.  There is no CPU fallback: if the library
cannot be loaded, or no CUDA device is usable, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass, field
from typing import Any, Optional

import numpy as np

__all__ = ["gtls_search", "gtls_search_static", "gtls_static_scratch_bytes", "gtls_search_two_stage", "gtls_search_batch", "gtls_batch_workspace_bytes",
           "gtls_period_grid_size", "gtls_period_grid", "gtls_duration_grid", "BatchResult", "gtls_search_sharded", "gtls_fold_sort", "gtls_fold_scan", "gtls_window_chi2", "gtls_ring_window_chi2", "gtls_sde",
           "gtls_workspace_bytes", "gtls_release_cache", "gtls_peak_fp64", "gtls_strerror", "gtls_version", "GtlsError", "SearchResult",
           "BEST_DTYPE", "lib_path", "load_library"]

_PKG = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_PKG, "libgtls.so")

GTLS_OK = 0
GTLS_EDEGENERATE = -6

BEST_DTYPE = np.dtype([("dur_idx", np.int32), ("start", np.int32), ("depth", np.float64),
                       ("t0", np.float64)], align=True)


class GtlsStats(C.Structure):
    _fields_ = [("ms_total", C.c_double), ("ms_pre", C.c_double), ("ms_fold", C.c_double),
                ("ms_sort", C.c_double), ("ms_scan", C.c_double), ("ms_chi2", C.c_double),
                ("ms_reduce", C.c_double), ("ms_epilogue", C.c_double),
                ("kernel_launches", C.c_int64), ("chi2_launches", C.c_int64),
                ("windows", C.c_int64), ("window_points", C.c_int64), ("period_points", C.c_int64),
                ("period_tile", C.c_int32), ("path", C.c_int32), ("uniform_dy", C.c_int32),
                ("reserved", C.c_int32)]

    def as_dict(self) -> dict:
        return {k: getattr(self, k) for k, _ in self._fields_ if k != "reserved"}


class GtlsOpts(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("dt0", C.c_double), ("top_k", C.c_int32),
                ("dur_per_period", C.c_int32), ("sde_kernel", C.c_int32), ("chi2_fp32", C.c_int32),
                ("pointers_on_device", C.c_int32), ("device", C.c_int32), ("stream", C.c_void_p),
                ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
                ("period_tile", C.c_int32), ("path", C.c_int32), ("stats", C.POINTER(GtlsStats))]


class GtlsSummary(C.Structure):
    _fields_ = [("best_period_idx", C.c_int64), ("best_dur_idx", C.c_int32), ("best_start", C.c_int32),
                ("best_period", C.c_double), ("best_t0", C.c_double), ("best_depth", C.c_double),
                ("chi2_min", C.c_double), ("chi2_null", C.c_double), ("sde_raw_max", C.c_double),
                ("sde_max", C.c_double), ("sde_argmax", C.c_int64), ("windows_evaluated", C.c_int64)]

    def as_dict(self) -> dict:
        return {k: getattr(self, k) for k, _ in self._fields_}


class GtlsError(RuntimeError):
    def __init__(self, code: int, where: str):
        lib = load_library()
        msg = lib.gtls_strerror(code).decode()
        cuda = lib.gtls_last_cuda_error().decode()
        super().__init__(f"{where}: {msg} [{code}]" + (f" -- {cuda}" if cuda else ""))
        self.code = code


_lib = None


def lib_path() -> str:
    return _LIB_PATH


def load_library():
    """Load libgtls.so (built in-tree by ``python -m paper_2607_00348_b200.build``).  Raises if it
    is missing: there is deliberately no fallback implementation."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError(f"{_LIB_PATH} not found: build it with "
                          "`python -m paper_2607_00348_b200.build` (nvcc, sm_100a); "
                          "there is no CPU fallback")
    lib = C.CDLL(_LIB_PATH)
    vp, dp, ip = C.c_void_p, C.c_void_p, C.c_void_p
    lib.gtls_opts_default.argtypes = [C.POINTER(GtlsOpts)]
    lib.gtls_opts_default.restype = None
    lib.gtls_search.argtypes = [dp, dp, dp, C.c_int64, dp, C.c_int64, dp, C.c_int32, dp, C.c_int32,
                                C.POINTER(GtlsOpts), dp, vp, dp, dp, C.POINTER(GtlsSummary)]
    lib.gtls_search.restype = C.c_int
    lib.gtls_search_static.argtypes = lib.gtls_search.argtypes
    lib.gtls_search_static.restype = C.c_int
    lib.gtls_static_scratch_bytes.argtypes = []
    lib.gtls_static_scratch_bytes.restype = C.c_size_t
    lib.gtls_search_two_stage.argtypes = [dp, dp, dp, C.c_int64, dp, C.c_int64, dp, C.c_int32, dp, C.c_int32,
                                          C.POINTER(GtlsOpts), C.c_int32, dp, vp, dp, dp, vp,
                                          C.POINTER(GtlsSummary)]
    lib.gtls_search_two_stage.restype = C.c_int
    lib.gtls_fold_sort.argtypes = [dp, C.c_int64, dp, C.c_int64, C.POINTER(GtlsOpts), dp, ip]
    lib.gtls_fold_sort.restype = C.c_int
    lib.gtls_fold_scan.argtypes = [dp, dp, dp, C.c_int64, C.c_double, C.c_int64, C.POINTER(GtlsOpts),
                                   dp, dp, dp]
    lib.gtls_fold_scan.restype = C.c_int
    lib.gtls_window_chi2.argtypes = [dp, dp, dp, C.c_int64, C.c_double, C.c_double, dp, C.c_int32,
                                     C.POINTER(GtlsOpts), ip, dp, dp, dp]
    lib.gtls_window_chi2.restype = C.c_int64
    lib.gtls_ring_window_chi2.argtypes = [dp, dp, dp, C.c_int64, C.c_double, C.c_double, dp, C.c_int32,
                                          C.POINTER(GtlsOpts), ip, dp, dp, C.POINTER(C.c_double)]
    lib.gtls_ring_window_chi2.restype = C.c_int64
    lib.gtls_sde.argtypes = [dp, C.c_int64, C.POINTER(GtlsOpts), dp, dp, C.POINTER(GtlsSummary)]
    lib.gtls_sde.restype = C.c_int
    lib.gtls_period_grid_size.argtypes = [C.c_double] * 5
    lib.gtls_period_grid_size.restype = C.c_int64
    lib.gtls_period_grid.argtypes = [C.c_double] * 5 + [C.POINTER(GtlsOpts), dp, C.c_int64]
    lib.gtls_period_grid.restype = C.c_int
    lib.gtls_duration_grid.argtypes = [dp, C.c_int64, C.c_int32, C.c_double, C.c_double, C.c_double,
                                       C.POINTER(GtlsOpts), dp]
    lib.gtls_duration_grid.restype = C.c_int
    lib.gtls_search_batch.argtypes = [C.c_int32, dp, dp, dp, vp, dp, vp, dp, C.c_int32, dp, C.c_int32,
                                      C.POINTER(GtlsOpts), dp, vp, dp, dp, vp, vp]
    lib.gtls_search_batch.restype = C.c_int
    lib.gtls_batch_workspace_bytes.argtypes = [C.c_int32, vp, vp, C.c_int32, C.POINTER(GtlsOpts)]
    lib.gtls_batch_workspace_bytes.restype = C.c_size_t
    lib.gtls_workspace_bytes.argtypes = [C.c_int64, C.c_int64, C.c_int32, C.POINTER(GtlsOpts)]
    lib.gtls_workspace_bytes.restype = C.c_size_t
    lib.gtls_peak_fp64.argtypes = [C.c_double, C.POINTER(GtlsOpts), C.POINTER(C.c_double), C.POINTER(C.c_double),
                                   C.POINTER(C.c_int64)]
    lib.gtls_peak_fp64.restype = C.c_int
    lib.gtls_release_cache.argtypes = []
    lib.gtls_release_cache.restype = None
    lib.gtls_strerror.argtypes = [C.c_int]
    lib.gtls_strerror.restype = C.c_char_p
    lib.gtls_version.restype = C.c_char_p
    lib.gtls_last_cuda_error.restype = C.c_char_p
    _lib = lib
    return lib


# ---------------------------------------------------------------------------------------------
# marshalling helpers
# ---------------------------------------------------------------------------------------------
def _is_torch(x) -> bool:
    return type(x).__module__.startswith("torch")


def _prep(x, dtype=np.float64):
    """Return (object kept alive, pointer int, is_device)."""
    if _is_torch(x):
        import torch
        want = {np.float64: torch.float64, np.int32: torch.int32}[dtype]
        if not x.is_cuda:
            raise ValueError("torch inputs must be CUDA tensors (use numpy arrays for host data)")
        x = x.contiguous()
        if x.dtype != want:
            x = x.to(want)
        return x, x.data_ptr(), True
    a = np.ascontiguousarray(x, dtype=dtype)
    return a, a.ctypes.data, False


def _opts(device_mode: bool, like=None, stream=None, **kw) -> GtlsOpts:
    o = GtlsOpts()
    load_library().gtls_opts_default(C.byref(o))
    o.pointers_on_device = 1 if device_mode else 0
    if device_mode:
        import torch
        o.device = like.device.index if like.device.index is not None else torch.cuda.current_device()
        s = stream if stream is not None else torch.cuda.current_stream(like.device)
        o.stream = int(getattr(s, "cuda_stream", s))
    for k, v in kw.items():
        setattr(o, k, v)
    return o


def _empty(shape, like, dtype=np.float64):
    if _is_torch(like):
        import torch
        td = {np.float64: torch.float64, np.int32: torch.int32, np.uint8: torch.uint8}[dtype]
        return torch.empty(shape, dtype=td, device=like.device)
    return np.empty(shape, dtype=dtype)


def _ptr(x) -> int:
    return x.data_ptr() if _is_torch(x) else x.ctypes.data


# ---------------------------------------------------------------------------------------------
# entry points (same names as include/gtls.h)
# ---------------------------------------------------------------------------------------------
@dataclass
class SearchResult:
    chi2: Any                      # [n_per]
    sde_raw: Any                   # [n_per]
    sde: Any                       # [n_per]
    best_raw: Any                  # [n_per, 24] bytes: gtls_best records
    summary: dict
    code: int                      # GTLS_OK or GTLS_EDEGENERATE
    stats: Optional[dict] = None
    _keep: list = field(default_factory=list, repr=False)

    def best(self) -> np.ndarray:
        """gtls_best records as a numpy structured array (copies from the device)."""
        raw = self.best_raw.cpu().numpy() if _is_torch(self.best_raw) else self.best_raw
        return np.ascontiguousarray(raw).view(BEST_DTYPE).reshape(-1)


def gtls_version() -> str:
    return load_library().gtls_version().decode()


def gtls_release_cache() -> None:
    """Free the device blocks the library keeps between calls (``gtls_release_cache`` in include/gtls.h)."""
    load_library().gtls_release_cache()


def gtls_peak_fp64(seconds: float, device: int = 0, stream: int = 0) -> dict:
    """fp64 FMA microbenchmark (``gtls_peak_fp64`` in include/gtls.h): sustained TFLOP/s over `seconds`."""
    lib = load_library()
    o = GtlsOpts()
    lib.gtls_opts_default(C.byref(o))
    o.device = int(device)
    o.stream = int(stream)
    tf, ms, nl = C.c_double(0.0), C.c_double(0.0), C.c_int64(0)
    rc = lib.gtls_peak_fp64(float(seconds), C.byref(o), C.byref(tf), C.byref(ms), C.byref(nl))
    if rc != GTLS_OK:
        raise GtlsError(rc, "gtls_peak_fp64")
    return {"tflops": tf.value, "ms": ms.value, "launches": nl.value}


def gtls_strerror(code: int) -> str:
    return load_library().gtls_strerror(int(code)).decode()


def gtls_workspace_bytes(n: int, n_per: int, n_dur: int, period_tile: int = 0) -> int:
    o = GtlsOpts()
    lib = load_library()
    lib.gtls_opts_default(C.byref(o))
    o.period_tile = int(period_tile)
    return int(lib.gtls_workspace_bytes(int(n), int(n_per), int(n_dur), C.byref(o)))


def gtls_search(t, y, dy, period_grid, duration_grid, tmpl, *, dt0: float = 0.05,
                sde_kernel: int = 151, top_k: int = 0, chi2_fp32: int = 0, period_tile: int = 0,
                path: int = 0, workspace=None, stats: bool = False, stream=None) -> SearchResult:
    """TLS period search (``gtls_search`` in include/gtls.h).  ``duration_grid`` is [n_dur]
    (shared) or [n_per, n_dur] (one row per period)."""
    lib = load_library()
    kt, pt, dev = _prep(t)
    ky, py, d2 = _prep(y)
    kd, pd, d3 = _prep(dy)
    kp, pp, d4 = _prep(period_grid)
    kq, pq, d5 = _prep(duration_grid)
    km, pm, d6 = _prep(tmpl)
    if len({dev, d2, d3, d4, d5, d6}) != 1:
        raise ValueError("all arrays must be either CUDA tensors or host arrays")
    n, n_per, n_tmpl = int(kt.shape[0]), int(kp.shape[0]), int(km.shape[0])
    per_period = 1 if kq.ndim == 2 else 0
    n_dur = int(kq.shape[-1])
    if per_period and int(kq.shape[0]) != n_per:
        raise ValueError("duration_grid rows must match period_grid")
    st = GtlsStats()
    o = _opts(dev, kt, stream, dt0=float(dt0), sde_kernel=int(sde_kernel), top_k=int(top_k),
              chi2_fp32=int(chi2_fp32), dur_per_period=per_period, period_tile=int(period_tile),
              path=int(path))
    if stats:
        o.stats = C.pointer(st)
    if workspace is not None:
        if not (_is_torch(workspace) and workspace.is_cuda):
            raise ValueError("workspace must be a CUDA uint8 tensor")
        o.workspace = workspace.data_ptr()
        o.workspace_bytes = workspace.numel() * workspace.element_size()
    chi2 = _empty((n_per,), kt)
    sde_raw = _empty((n_per,), kt)
    sde = _empty((n_per,), kt)
    best = _empty((n_per, BEST_DTYPE.itemsize), kt, np.uint8)
    summ = GtlsSummary()
    rc = lib.gtls_search(pt, py, pd, n, pp, n_per, pq, n_dur, pm, n_tmpl, C.byref(o), _ptr(chi2),
                         _ptr(best), _ptr(sde_raw), _ptr(sde), C.byref(summ))
    if rc not in (GTLS_OK, GTLS_EDEGENERATE):
        raise GtlsError(rc, "gtls_search")
    return SearchResult(chi2, sde_raw, sde, best, summ.as_dict(), rc,
                        st.as_dict() if stats else None, [kt, ky, kd, kp, kq, km])


def gtls_search_static(t, y, dy, period_grid, duration_grid, tmpl, *, dt0: float = 0.05, sde_kernel: int = 151,
                       out=None, stream=None) -> SearchResult:
    """The allocation-free search (``gtls_search_static`` in include/gtls.h): CUDA tensors only; the library
    uses its static scratch array and allocates nothing.  ``out`` = (chi2, best_raw, sde_raw, sde) tensors to
    write into (float64[n_per], uint8[n_per, 24], float64[n_per] x 2); created here when None."""
    lib = load_library()
    kt, pt, dev = _prep(t)
    ky, py, d2 = _prep(y)
    kd, pd, d3 = _prep(dy)
    kp, pp, d4 = _prep(period_grid)
    kq, pq, d5 = _prep(duration_grid)
    km, pm, d6 = _prep(tmpl)
    if not all((dev, d2, d3, d4, d5, d6)):
        raise ValueError("gtls_search_static takes CUDA tensors only")
    n, n_per, n_tmpl = int(kt.shape[0]), int(kp.shape[0]), int(km.shape[0])
    per_period = 1 if kq.ndim == 2 else 0
    n_dur = int(kq.shape[-1])
    if per_period and int(kq.shape[0]) != n_per:
        raise ValueError("duration_grid rows must match period_grid")
    o = _opts(True, kt, stream, dt0=float(dt0), sde_kernel=int(sde_kernel), dur_per_period=per_period)
    if out is None:
        out = (_empty((n_per,), kt), _empty((n_per, BEST_DTYPE.itemsize), kt, np.uint8), _empty((n_per,), kt),
               _empty((n_per,), kt))
    chi2, best, sde_raw, sde = out
    summ = GtlsSummary()
    rc = lib.gtls_search_static(pt, py, pd, n, pp, n_per, pq, n_dur, pm, n_tmpl, C.byref(o), _ptr(chi2),
                                _ptr(best), _ptr(sde_raw), _ptr(sde), C.byref(summ))
    if rc not in (GTLS_OK, GTLS_EDEGENERATE):
        raise GtlsError(rc, "gtls_search_static")
    return SearchResult(chi2, sde_raw, sde, best, summ.as_dict(), rc, None, [kt, ky, kd, kp, kq, km])


def gtls_static_scratch_bytes() -> int:
    return int(load_library().gtls_static_scratch_bytes())


def gtls_period_grid_size(span: float, r_star: float = 1.0, m_star: float = 1.0, oversampling: float = 3.0,
                          p_min: float = 0.0) -> int:
    """N = ceil(Eq. 6) of the Ofir period grid (``gtls_period_grid_size`` in include/gtls.h)."""
    n = int(load_library().gtls_period_grid_size(float(span), float(r_star), float(m_star),
                                                  float(oversampling), float(p_min)))
    if n < 0:
        raise GtlsError(n, "gtls_period_grid_size")
    return n


def gtls_period_grid(span: float, r_star: float = 1.0, m_star: float = 1.0, oversampling: float = 3.0,
                     p_min: float = 0.0, *, device=None, stream=None):
    """Ofir period grid (Eq. 1-6) built on the device.  ``device`` = a torch CUDA device: the result is
    a CUDA tensor; ``None``: a numpy array (the library copies it back)."""
    lib = load_library()
    args = (float(span), float(r_star), float(m_star), float(oversampling), float(p_min))
    n = gtls_period_grid_size(*args)
    if device is not None:
        import torch
        out = torch.empty(n, dtype=torch.float64, device=device)
        o = _opts(True, out, stream)
    else:
        out = np.empty(n, dtype=np.float64)
        o = _opts(False)
    rc = lib.gtls_period_grid(*args, C.byref(o), _ptr(out), n)
    if rc != GTLS_OK:
        raise GtlsError(rc, "gtls_period_grid")
    return out


def gtls_duration_grid(periods, n_dur: int, k_min: float = 20.05, k_max: float = 620.84,
                       q_cap: float = 0.15, *, stream=None):
    """[n_per, n_dur] duration fractions T14/P (Eq. 8-9 + cap, reading G12) built on the device."""
    lib = load_library()
    kp, pp, dev = _prep(periods)
    n_per = int(kp.shape[0])
    out = _empty((n_per, int(n_dur)), kp)
    o = _opts(dev, kp, stream)
    rc = lib.gtls_duration_grid(pp, n_per, int(n_dur), float(k_min), float(k_max), float(q_cap),
                                C.byref(o), _ptr(out))
    if rc != GTLS_OK:
        raise GtlsError(rc, "gtls_duration_grid")
    return out


@dataclass
class BatchResult:
    chi2: Any                      # [total periods], curve after curve
    sde_raw: Any
    sde: Any
    best_raw: Any                  # [total periods, 24] bytes
    period_offset: np.ndarray      # [n_curves + 1]
    summaries: list                # one dict per curve
    status: np.ndarray             # [n_curves] int32: GTLS_OK / GTLS_EDEGENERATE per curve
    _keep: list = field(default_factory=list, repr=False)

    def best(self) -> np.ndarray:
        raw = self.best_raw.cpu().numpy() if _is_torch(self.best_raw) else self.best_raw
        return np.ascontiguousarray(raw).view(BEST_DTYPE).reshape(-1)


def _offsets(x, name: str) -> np.ndarray:
    a = np.ascontiguousarray(np.asarray(x.cpu() if _is_torch(x) else x), dtype=np.int64)
    if a.ndim != 1 or a.size < 2:
        raise ValueError(f"{name} must hold n_curves + 1 entries")
    return a


def gtls_batch_workspace_bytes(curve_offset, period_offset, n_dur: int, period_tile: int = 0) -> int:
    co, po = _offsets(curve_offset, "curve_offset"), _offsets(period_offset, "period_offset")
    o = GtlsOpts()
    lib = load_library()
    lib.gtls_opts_default(C.byref(o))
    o.period_tile = int(period_tile)
    return int(lib.gtls_batch_workspace_bytes(co.size - 1, co.ctypes.data, po.ctypes.data, int(n_dur), C.byref(o)))


def gtls_search_batch(t, y, dy, curve_offset, period_grid, period_offset, duration_grid, tmpl, *,
                      dt0: float = 0.05, sde_kernel: int = 151, top_k: int = 0, chi2_fp32: int = 0,
                      period_tile: int = 0, path: int = 0, workspace=None, stream=None) -> BatchResult:
    """Survey mode (``gtls_search_batch`` in include/gtls.h): concatenated light curves and period
    grids with host offset arrays; ``duration_grid`` is [n_dur] (shared) or [total periods, n_dur]."""
    lib = load_library()
    co, po = _offsets(curve_offset, "curve_offset"), _offsets(period_offset, "period_offset")
    if co.size != po.size:
        raise ValueError("curve_offset and period_offset must have the same length")
    n_curves = co.size - 1
    kt, pt, dev = _prep(t)
    ky, py, d2 = _prep(y)
    kd, pd, d3 = _prep(dy)
    kp, pp, d4 = _prep(period_grid)
    kq, pq, d5 = _prep(duration_grid)
    km, pm, d6 = _prep(tmpl)
    if len({dev, d2, d3, d4, d5, d6}) != 1:
        raise ValueError("all arrays must be either CUDA tensors or host arrays")
    if int(kt.shape[0]) != int(co[-1]) or int(kp.shape[0]) != int(po[-1]):
        raise ValueError("offsets do not match the array lengths")
    per_total, n_tmpl = int(po[-1]), int(km.shape[0])
    per_period = 1 if kq.ndim == 2 else 0
    n_dur = int(kq.shape[-1])
    if per_period and int(kq.shape[0]) != per_total:
        raise ValueError("duration_grid rows must match period_grid")
    o = _opts(dev, kt, stream, dt0=float(dt0), sde_kernel=int(sde_kernel), top_k=int(top_k),
              chi2_fp32=int(chi2_fp32), dur_per_period=per_period, period_tile=int(period_tile), path=int(path))
    if workspace is not None:
        if not (_is_torch(workspace) and workspace.is_cuda):
            raise ValueError("workspace must be a CUDA uint8 tensor")
        o.workspace = workspace.data_ptr()
        o.workspace_bytes = workspace.numel() * workspace.element_size()
    chi2 = _empty((per_total,), kt)
    sde_raw = _empty((per_total,), kt)
    sde = _empty((per_total,), kt)
    best = _empty((per_total, BEST_DTYPE.itemsize), kt, np.uint8)
    summ = (GtlsSummary * n_curves)()
    status = np.zeros(n_curves, dtype=np.int32)
    rc = lib.gtls_search_batch(n_curves, pt, py, pd, co.ctypes.data, pp, po.ctypes.data, pq, n_dur, pm, n_tmpl,
                               C.byref(o), _ptr(chi2), _ptr(best), _ptr(sde_raw), _ptr(sde),
                               C.cast(summ, C.c_void_p), status.ctypes.data)
    if rc != GTLS_OK:
        raise GtlsError(rc, "gtls_search_batch")
    return BatchResult(chi2, sde_raw, sde, best, po, [s_.as_dict() for s_ in summ], status,
                       [kt, ky, kd, kp, kq, km])


def gtls_search_two_stage(t, y, dy, period_grid, duration_grid, tmpl, *, dt0: float = 0.05,
                          n_refine: int = 200, sde_kernel: int = 151, period_tile: int = 0, workspace=None,
                          stream=None):
    """Two-stage hierarchical search (``gtls_search_two_stage`` in include/gtls.h): returns
    (SearchResult, refined) with ``refined`` the int64 indices of the refined periods."""
    lib = load_library()
    kt, pt, dev = _prep(t)
    ky, py, d2 = _prep(y)
    kd, pd, d3 = _prep(dy)
    kp, pp, d4 = _prep(period_grid)
    kq, pq, d5 = _prep(duration_grid)
    km, pm, d6 = _prep(tmpl)
    if len({dev, d2, d3, d4, d5, d6}) != 1:
        raise ValueError("all arrays must be either CUDA tensors or host arrays")
    n, n_per, n_tmpl = int(kt.shape[0]), int(kp.shape[0]), int(km.shape[0])
    per_period = 1 if kq.ndim == 2 else 0
    n_dur = int(kq.shape[-1])
    o = _opts(dev, kt, stream, dt0=float(dt0), sde_kernel=int(sde_kernel), dur_per_period=per_period,
              period_tile=int(period_tile))
    if workspace is not None:
        o.workspace = workspace.data_ptr()
        o.workspace_bytes = workspace.numel() * workspace.element_size()
    chi2 = _empty((n_per,), kt)
    sde_raw = _empty((n_per,), kt)
    sde = _empty((n_per,), kt)
    best = _empty((n_per, BEST_DTYPE.itemsize), kt, np.uint8)
    k = min(int(n_refine), n_per)
    if _is_torch(kt):
        import torch
        refined = torch.empty((max(k, 1),), dtype=torch.int64, device=kt.device)
    else:
        refined = np.empty((max(k, 1),), dtype=np.int64)
    summ = GtlsSummary()
    rc = lib.gtls_search_two_stage(pt, py, pd, n, pp, n_per, pq, n_dur, pm, n_tmpl, C.byref(o), int(n_refine),
                                   _ptr(chi2), _ptr(best), _ptr(sde_raw), _ptr(sde), _ptr(refined),
                                   C.byref(summ))
    if rc not in (GTLS_OK, GTLS_EDEGENERATE):
        raise GtlsError(rc, "gtls_search_two_stage")
    res = SearchResult(chi2, sde_raw, sde, best, summ.as_dict(), rc, None, [kt, ky, kd, kp, kq, km])
    return res, refined[:k]


def gtls_fold_sort(t, periods, *, want_phase: bool = True, period_tile: int = 0, stream=None):
    """Phases (Eq. 10) and stable phase-sort permutations for each period: (phase, perm)."""
    lib = load_library()
    kt, pt, dev = _prep(t)
    kp, pp, d2 = _prep(periods)
    if dev != d2:
        raise ValueError("all arrays must be either CUDA tensors or host arrays")
    n, n_per = int(kt.shape[0]), int(kp.shape[0])
    o = _opts(dev, kt, stream, period_tile=int(period_tile))
    phase = _empty((n_per, n), kt) if want_phase else None
    perm = _empty((n_per, n), kt, np.int32)
    rc = lib.gtls_fold_sort(pt, n, pp, n_per, C.byref(o), _ptr(phase) if want_phase else None, _ptr(perm))
    if rc != GTLS_OK:
        raise GtlsError(rc, "gtls_fold_sort")
    return phase, perm


def gtls_fold_scan(t, y, dy, period: float, pad: int, *, stream=None):
    """Wrap-padded prefix sums (S1 of w r, S0 of w, S2 of w r^2) for one period, each of
    length n + pad + 1."""
    lib = load_library()
    kt, pt, dev = _prep(t)
    ky, py, d2 = _prep(y)
    kd, pd, d3 = _prep(dy)
    if len({dev, d2, d3}) != 1:
        raise ValueError("all arrays must be either CUDA tensors or host arrays")
    n = int(kt.shape[0])
    o = _opts(dev, kt, stream)
    outs = [_empty((n + int(pad) + 1,), kt) for _ in range(3)]
    rc = lib.gtls_fold_scan(pt, py, pd, n, float(period), int(pad), C.byref(o), *[_ptr(x) for x in outs])
    if rc != GTLS_OK:
        raise GtlsError(rc, "gtls_fold_scan")
    return tuple(outs)


def gtls_window_chi2(t, y, dy, period: float, q: float, tmpl, *, dt0: float = 0.0, stream=None):
    """Per-window terms for one (period, duration fraction): (start, depth, chi2_out, chi2_in)."""
    lib = load_library()
    kt, pt, dev = _prep(t)
    ky, py, d2 = _prep(y)
    kd, pd, d3 = _prep(dy)
    km, pm, d4 = _prep(tmpl)
    if len({dev, d2, d3, d4}) != 1:
        raise ValueError("all arrays must be either CUDA tensors or host arrays")
    n = int(kt.shape[0])
    o = _opts(dev, kt, stream, dt0=float(dt0))
    start = _empty((n,), kt, np.int32)
    depth, c_out, c_in = (_empty((n,), kt) for _ in range(3))
    k = lib.gtls_window_chi2(pt, py, pd, n, float(period), float(q), pm, int(km.shape[0]), C.byref(o),
                             _ptr(start), _ptr(depth), _ptr(c_out), _ptr(c_in))
    if k < 0:
        raise GtlsError(int(k), "gtls_window_chi2")
    k = int(k)
    return start[:k], depth[:k], c_out[:k], c_in[:k]


def gtls_ring_window_chi2(t, y, dy, period: float, q: float, tmpl, *, dt0: float = 0.0, path: int = 2):
    """Every window of one (period, duration fraction) as the hot kernel scores it (``gtls_ring_window_chi2`` in
    include/gtls.h; host arrays): (start, depth, dchi2, chi2_null).  path = 2: the ring kernel of the general
    path; path = 1: the fused small-N kernel."""
    lib = load_library()
    t, y, dy, tmpl = (np.ascontiguousarray(a, dtype=np.float64) for a in (t, y, dy, tmpl))
    n = int(t.shape[0])
    o = GtlsOpts()
    lib.gtls_opts_default(C.byref(o))
    o.dt0 = float(dt0)
    o.path = int(path)
    start = np.empty(n, dtype=np.int32)
    depth, dchi2 = np.empty(n), np.empty(n)
    c0 = C.c_double(0.0)
    k = lib.gtls_ring_window_chi2(t.ctypes.data, y.ctypes.data, dy.ctypes.data, n, float(period), float(q),
                                  tmpl.ctypes.data, int(tmpl.shape[0]), C.byref(o), start.ctypes.data,
                                  depth.ctypes.data, dchi2.ctypes.data, C.byref(c0))
    if k < 0:
        raise GtlsError(int(k), "gtls_ring_window_chi2")
    k = int(k)
    return start[:k], depth[:k], dchi2[:k], c0.value


def gtls_sde(chi2, *, sde_kernel: int = 151, stream=None):
    """SR/SDE epilogue alone: returns (sde_raw, sde, summary dict, code)."""
    lib = load_library()
    kc, pc, dev = _prep(chi2)
    n_per = int(kc.shape[0])
    o = _opts(dev, kc, stream, sde_kernel=int(sde_kernel))
    raw = _empty((n_per,), kc)
    sde = _empty((n_per,), kc)
    summ = GtlsSummary()
    rc = lib.gtls_sde(pc, n_per, C.byref(o), _ptr(raw), _ptr(sde), C.byref(summ))
    if rc not in (GTLS_OK, GTLS_EDEGENERATE):
        raise GtlsError(rc, "gtls_sde")
    return raw, sde, summ.as_dict(), rc


def gtls_search_sharded(t, y, dy, period_grid, duration_grid, tmpl, *, group=None, dt0: float = 0.05,
                        sde_kernel: int = 151, **kw) -> SearchResult:
    """Period-sharded search over the ranks of a ``torch.distributed`` group (one process per GPU).

    Trial periods are independent (the paper reports 1.75x on two GPUs), so
    rank r searches periods r, r+W, r+2W, ... (interleaved: every rank gets the same mix of long and short
    periods, i.e. of durations), the only exchange is ONE all-gather of 32 bytes per period (chi2 + the
    24-byte best record), and every rank then runs the SR / SDE epilogue (``gtls_sde``) over the full
    spectrum in grid order.  Every rank passes the same full arrays and gets the same full result."""
    return _sharded_search(gtls_search, gtls_sde, t, y, dy, period_grid, duration_grid, tmpl, group=group, dt0=dt0,
                           sde_kernel=sde_kernel, **kw)


def _sharded_search(search, sde_fn, t, y, dy, period_grid, duration_grid, tmpl, *, group=None, dt0: float = 0.05,
                    sde_kernel: int = 151, **kw) -> SearchResult:
    """The plumbing of gtls_search_sharded around the two library calls (`search`, `sde_fn`); the CPU (gloo)
    test of the shard / all-gather / unshard logic calls this private helper with stand-ins for them."""
    import torch
    import torch.distributed as dist
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    n_per = int(period_grid.shape[0])
    per_period = duration_grid.ndim == 2
    mine = slice(rank, n_per, world)
    cont = (lambda a: a.contiguous()) if _is_torch(period_grid) else np.ascontiguousarray
    res = search(t, y, dy, cont(period_grid[mine]), cont(duration_grid[mine]) if per_period else duration_grid,
                 tmpl, dt0=dt0, sde_kernel=0, **kw)
    # ---- one all-gather: [m, 4] doubles per rank = chi2 + the best record's 24 bytes, padded to m rows ----
    m = (n_per + world - 1) // world
    on_gpu = _is_torch(res.chi2)
    comm_dev = res.chi2.device if (on_gpu and dist.get_backend(group) == "nccl") else torch.device("cpu")
    as_t = (lambda a: a) if on_gpu else (lambda a: torch.from_numpy(np.ascontiguousarray(a)))
    chi2_l = as_t(res.chi2).to(comm_dev)
    best_l = as_t(res.best_raw).to(comm_dev).contiguous().view(torch.float64).reshape(-1, 3)
    pack = torch.full((m, 4), float("inf"), dtype=torch.float64, device=comm_dev)
    pack[: chi2_l.shape[0], 0] = chi2_l
    pack[: chi2_l.shape[0], 1:] = best_l
    parts = [torch.empty_like(pack) for _ in range(world)]
    dist.all_gather(parts, pack, group=group)
    gathered = torch.stack(parts)                                        # [world, m, 4]
    nwin = torch.tensor([int(res.summary.get("windows_evaluated", 0))], dtype=torch.int64, device=comm_dev)
    dist.all_reduce(nwin, group=group)
    full = gathered.permute(1, 0, 2).reshape(world * m, 4)[:n_per]     # row i*W + r  <-  rank r's row i
    chi2 = full[:, 0].contiguous()
    best_raw = full[:, 1:].contiguous().view(torch.uint8).reshape(n_per, BEST_DTYPE.itemsize)
    if on_gpu:
        chi2, best_raw = chi2.to(res.chi2.device), best_raw.to(res.chi2.device)
    else:
        chi2, best_raw = chi2.numpy(), best_raw.numpy()
    sde_raw, sde, summ, rc = sde_fn(chi2, sde_kernel=sde_kernel)
    # the epilogue knows chi2 only: fill the best-period fields from the gathered records
    ib = int(summ["best_period_idx"])
    rec = (best_raw[ib].cpu().numpy() if _is_torch(best_raw) else best_raw[ib]).view(BEST_DTYPE)[0]
    summ = dict(summ, best_period=float(period_grid[ib]), best_dur_idx=int(rec["dur_idx"]),
                best_start=int(rec["start"]), best_depth=float(rec["depth"]), best_t0=float(rec["t0"]),
                chi2_null=res.summary.get("chi2_null", 0.0), windows_evaluated=int(nwin.item()))
    return SearchResult(chi2, sde_raw, sde, best_raw, summ, rc, None, [res])
