"""CPU oracle for the TLS/GTLS period search -- TEST INFRASTRUCTURE, not the product.

Thin ctypes binding over ``oracle/gtls_oracle.cpp`` (see that file's header for the
citations, readings and pins).  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import this package; the
product path (``paper_2607_00348_b200``) never does.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass

import numpy as np

from . import build as _build

_lib = None


class _Best(C.Structure):
    _fields_ = [("dur_idx", C.c_int32), ("start", C.c_int32), ("depth", C.c_double), ("t0", C.c_double)]


BEST_DTYPE = np.dtype([("dur_idx", np.int32), ("start", np.int32), ("depth", np.float64),
                       ("t0", np.float64)], align=True)

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_lp = C.POINTER(C.c_int64)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.oracle_num_threads.restype = C.c_int
        _lib.oracle_points_in_duration.restype = C.c_int64
        _lib.oracle_points_in_duration.argtypes = [C.c_double, C.c_int64]
        _lib.oracle_stride.restype = C.c_int64
        _lib.oracle_stride.argtypes = [C.c_int64, C.c_double]
        _lib.oracle_resample_template.restype = C.c_double
        _lib.oracle_resample_template.argtypes = [_dp, C.c_int32, C.c_int64, _dp]
        _lib.oracle_chi2_null.restype = C.c_double
        _lib.oracle_chi2_null.argtypes = [_dp, _dp, C.c_int64]
        _lib.oracle_fold.argtypes = [_dp, C.c_int64, C.c_double, _dp]
        _lib.oracle_fold_sort.argtypes = [_dp, C.c_int64, _dp, C.c_int64, _dp, _ip]
        _lib.oracle_window_chi2_literal.restype = C.c_int64
        _lib.oracle_window_chi2_literal.argtypes = [_dp, _dp, _dp, C.c_int64, C.c_double, C.c_double,
                                                    _dp, C.c_int32, C.c_double, _ip, _dp, _dp, _dp]
        _lib.oracle_search.restype = C.c_int
        _lib.oracle_search.argtypes = [_dp, _dp, _dp, C.c_int64, _dp, C.c_int64, _dp, C.c_int32,
                                       C.c_int32, _dp, C.c_int32, C.c_double, C.c_int32, C.c_int32,
                                       _dp, C.c_void_p, _dp, _lp]
        _lib.oracle_roche_fmax_hz.restype = C.c_double
        _lib.oracle_roche_fmax_hz.argtypes = [C.c_double, C.c_double]
        _lib.oracle_period_grid_size.restype = C.c_int64
        _lib.oracle_period_grid_size.argtypes = [C.c_double] * 5
        _lib.oracle_period_grid.restype = C.c_int64
        _lib.oracle_period_grid.argtypes = [C.c_double] * 5 + [_dp, C.c_int64]
        _lib.oracle_duration_grid.restype = None
        _lib.oracle_duration_grid.argtypes = [_dp, C.c_int64, C.c_int32, C.c_double, C.c_double, C.c_double, _dp]
        _lib.oracle_sde.restype = C.c_int
        _lib.oracle_sde.argtypes = [_dp, C.c_int64, C.c_int32, _dp, _dp, _dp, _lp, _lp]
    return _lib


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_dp)


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def roche_fmax_hz(r_star: float = 1.0, m_star: float = 1.0) -> float:
    """Eq. 3."""
    return float(lib().oracle_roche_fmax_hz(float(r_star), float(m_star)))


def period_grid(span_days: float, r_star: float = 1.0, m_star: float = 1.0, oversampling: float = 3.0,
                p_min_days: float = 0.0) -> np.ndarray:
    """Ofir cubic frequency sampling, Eq. 1-6; periods in days, longest first."""
    args = (float(span_days), float(r_star), float(m_star), float(oversampling), float(p_min_days))
    n = int(lib().oracle_period_grid_size(*args))
    out = np.empty(n, dtype=np.float64)
    got = int(lib().oracle_period_grid(*args, out.ctypes.data_as(_dp), n))
    assert got == n
    return out


def duration_grid(periods_days, n_dur: int, k_min: float = 20.05, k_max: float = 620.84,
                  q_cap: float = 0.15) -> np.ndarray:
    """[n_per, n_dur] fractions T14/P, Eq. 8-9 + cap, log-spaced (G12)."""
    p, pp = _d(periods_days)
    out = np.empty((p.size, int(n_dur)), dtype=np.float64)
    lib().oracle_duration_grid(pp, p.size, int(n_dur), float(k_min), float(k_max), float(q_cap),
                               out.ctypes.data_as(_dp))
    return out


def points_in_duration(q: float, n: int) -> int:
    return int(lib().oracle_points_in_duration(float(q), int(n)))


def stride(d: int, dt0: float) -> int:
    return int(lib().oracle_stride(int(d), float(dt0)))


def resample_template(tmpl, d: int):
    tmpl, tp = _d(tmpl)
    g = np.empty(int(d), dtype=np.float64)
    gbar = lib().oracle_resample_template(tp, tmpl.size, int(d), g.ctypes.data_as(_dp))
    return g, float(gbar)


def chi2_null(y, dy) -> float:
    y, yp = _d(y)
    dy, dp = _d(dy)
    return float(lib().oracle_chi2_null(yp, dp, y.size))


def fold(t, period: float) -> np.ndarray:
    t, tp = _d(t)
    out = np.empty_like(t)
    lib().oracle_fold(tp, t.size, float(period), out.ctypes.data_as(_dp))
    return out


def fold_sort(t, periods, want_phase: bool = True):
    t, tp = _d(t)
    periods, pp = _d(np.atleast_1d(periods))
    n, n_per = t.size, periods.size
    perm = np.empty((n_per, n), dtype=np.int32)
    phase = np.empty((n_per, n), dtype=np.float64) if want_phase else None
    lib().oracle_fold_sort(tp, n, pp, n_per, phase.ctypes.data_as(_dp) if want_phase else None,
                           perm.ctypes.data_as(_ip))
    return phase, perm


def window_chi2_literal(t, y, dy, period: float, q: float, tmpl, dt0: float = 0.0):
    t, tp = _d(t); y, yp = _d(y); dy, dp = _d(dy); tmpl, mp = _d(tmpl)
    n = t.size
    start = np.empty(n, dtype=np.int32)
    depth = np.empty(n); c_out = np.empty(n); c_in = np.empty(n)
    k = lib().oracle_window_chi2_literal(tp, yp, dp, n, float(period), float(q), mp, tmpl.size,
                                         float(dt0), start.ctypes.data_as(_ip),
                                         depth.ctypes.data_as(_dp), c_out.ctypes.data_as(_dp),
                                         c_in.ctypes.data_as(_dp))
    return start[:k].copy(), depth[:k].copy(), c_out[:k].copy(), c_in[:k].copy()


@dataclass
class SearchResult:
    chi2: np.ndarray
    best: np.ndarray          # structured: dur_idx, start, depth, t0
    gap: np.ndarray           # runner-up dchi2 minus best dchi2 (distinct values)
    chi2_null: float
    windows: int


def search(t, y, dy, periods, durations, tmpl, dt0: float = 0.05, top_k: int = 0,
           n_threads: int = 0) -> SearchResult:
    t, tp = _d(t); y, yp = _d(y); dy, dp = _d(dy); tmpl, mp = _d(tmpl)
    periods, pp = _d(np.atleast_1d(periods))
    durations = np.ascontiguousarray(durations, dtype=np.float64)
    per_period = 1 if durations.ndim == 2 else 0
    if per_period:
        assert durations.shape[0] == periods.size
    n_dur = durations.shape[-1]
    n_per = periods.size
    chi2 = np.empty(n_per)
    gap = np.empty(n_per)
    best = np.zeros(n_per, dtype=BEST_DTYPE)
    assert best.itemsize == C.sizeof(_Best)
    windows = C.c_int64(0)
    rc = lib().oracle_search(tp, yp, dp, t.size, pp, n_per, durations.ctypes.data_as(_dp), n_dur,
                             per_period, mp, tmpl.size, float(dt0), int(top_k), int(n_threads),
                             chi2.ctypes.data_as(_dp), best.ctypes.data_as(C.c_void_p),
                             gap.ctypes.data_as(_dp), C.byref(windows))
    if rc != 0:
        raise ValueError(f"oracle_search rc={rc}")
    return SearchResult(chi2, best, gap, chi2_null(y, dy), int(windows.value))


@dataclass
class SdeResult:
    sr: np.ndarray
    sde_raw: np.ndarray
    sde: np.ndarray
    best_period_idx: int
    sde_argmax: int
    degenerate: bool


def sde(chi2, kernel: int = 151) -> SdeResult:
    chi2, cp = _d(chi2)
    n = chi2.size
    sr = np.empty(n); raw = np.empty(n); out = np.empty(n)
    ib = C.c_int64(0); im = C.c_int64(0)
    rc = lib().oracle_sde(cp, n, int(kernel), sr.ctypes.data_as(_dp), raw.ctypes.data_as(_dp),
                          out.ctypes.data_as(_dp), C.byref(ib), C.byref(im))
    return SdeResult(sr, raw, out, int(ib.value), int(im.value), bool(rc))


@dataclass
class TwoStageResult:
    chi2: np.ndarray
    best: np.ndarray
    sde: SdeResult
    refined: np.ndarray        # indices of the refined periods, in selection order
    coarse_sde: np.ndarray     # SDE after stage 1 (what the selection ranked)
    windows: int


def search_two_stage(t, y, dy, periods, durations, tmpl, dt0: float = 0.05, n_refine: int = 200,
                     sde_kernel: int = 151) -> TwoStageResult:
    """Two-stage hierarchical search, PAPER.md:293-295 (section 2.5), step by step:
    stage 1 = the search with the T0 skip of Eq. 18 over all periods; stage 2 = the n_refine periods of
    highest SDE (ties: lower index) searched again without skipping (stride 1); their chi2 / best replace
    the stage-1 values; SR / SDE are then recomputed over the whole grid."""
    periods = np.ascontiguousarray(np.atleast_1d(periods), dtype=np.float64)
    durations = np.ascontiguousarray(durations, dtype=np.float64)
    r1 = search(t, y, dy, periods, durations, tmpl, dt0=dt0)
    s1 = sde(r1.chi2, sde_kernel)
    k = min(int(n_refine), periods.size)
    order = np.argsort(-s1.sde, kind="stable")[:k]        # highest SDE first, ties keep the lower index
    dur2 = durations[order] if durations.ndim == 2 else np.tile(durations, (k, 1))
    r2 = search(t, y, dy, periods[order], dur2, tmpl, dt0=0.0)
    chi2 = r1.chi2.copy()
    best = r1.best.copy()
    chi2[order] = r2.chi2
    best[order] = r2.best
    return TwoStageResult(chi2, best, sde(chi2, sde_kernel), order.astype(np.int64), s1.sde,
                          r1.windows + r2.windows)
