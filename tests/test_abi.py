"""Host-side checks that need no GPU: the C-ABI library loads, exports every symbol that
include/gtls.h declares, its structs match the binding, and argument errors are reported
before any CUDA work."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_2607_00348_b200 as g

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2607_00348_b200 import build
    build.build()
    return g.load_library()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "gtls.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gtls_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    syms = _declared_symbols()
    assert {"gtls_search", "gtls_fold_sort", "gtls_fold_scan", "gtls_window_chi2", "gtls_sde",
            "gtls_workspace_bytes", "gtls_strerror", "gtls_version", "gtls_last_cuda_error",
            "gtls_opts_default", "gtls_period_grid_size", "gtls_period_grid", "gtls_duration_grid",
            "gtls_search_batch", "gtls_batch_workspace_bytes", "gtls_search_two_stage"} <= set(syms)
    for s in syms:
        assert hasattr(lib, s), s


def test_struct_layouts_match_header(lib):
    assert C.sizeof(g.GtlsOpts) == 80 and g.GtlsOpts.stats.offset == 72
    assert C.sizeof(g.GtlsSummary) == 88
    assert C.sizeof(g.GtlsStats) == 8 * 8 + 5 * 8 + 4 * 4
    assert g.BEST_DTYPE.itemsize == 24
    o = g.GtlsOpts()
    lib.gtls_opts_default(C.byref(o))
    assert o.struct_size == 80 and o.dt0 == 0.05 and o.sde_kernel == 151 and o.top_k == 0
    assert o.pointers_on_device == 0 and not o.workspace


def test_strerror_and_version(lib):
    assert g.gtls_version().startswith("gtls-b200")
    assert g.gtls_strerror(0) == "ok"
    for code in range(-7, 0):
        assert g.gtls_strerror(code) not in ("ok", "unknown error code")


def test_workspace_bytes_monotone(lib):
    a = g.gtls_workspace_bytes(4188, 10483, 25, period_tile=64)
    b = g.gtls_workspace_bytes(4188, 10483, 25, period_tile=128)
    assert 0 < a < b
    assert g.gtls_workspace_bytes(2, 10, 5) == 0          # n < 3 is invalid
    big = g.gtls_workspace_bytes(132247, 418562, 30)
    assert big < 26 << 30                                  # automatic tile keeps scratch bounded (24 GiB budget)


def test_argument_errors_before_cuda(lib):
    t = np.linspace(0, 10, 50); y = np.ones(50); dy = np.full(50, 1e-3)
    tm = np.ones(8); per = np.array([1.0, 2.0]); q = np.array([0.1])
    with pytest.raises(g.GtlsError) as e:
        g.gtls_search(t[:2], y[:2], dy[:2], per, q, tm)
    assert e.value.code == -1
    with pytest.raises(g.GtlsError) as e:
        g.gtls_search(t, y, dy, per, q, tm, sde_kernel=10)
    assert e.value.code == -1
    with pytest.raises(g.GtlsError) as e:
        g.gtls_search(t, y, dy, per, q, tm, top_k=9)            # pruning variant takes K <= 8
    assert e.value.code == -7
    with pytest.raises(g.GtlsError) as e:
        g.gtls_search(t, y, dy, per, q, tm, top_k=-1)
    assert e.value.code == -1
    with pytest.raises(g.GtlsError) as e:
        g.gtls_search(t, y, dy, per, q, tm, dt0=-0.1)
    assert e.value.code == -1


def test_no_cpu_fallback_without_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    t = np.linspace(0, 10, 50); y = np.ones(50); dy = np.full(50, 1e-3)
    with pytest.raises(g.GtlsError) as e:
        g.gtls_search(t, y, dy, np.array([1.0]), np.array([0.1]), np.ones(8))
    assert e.value.code == -5 and "cuda" in str(e.value).lower()


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2607_00348_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
                assert "liboracle" not in src, f


def test_period_grid_size_is_host_logic_and_matches_oracle():
    """N = ceil(Eq. 6) needs no GPU; the oracle computes it with its own code."""
    import oracle
    for span, kw in [(30.0, dict(p_min=0.5)), (90.0, dict(p_min=0.5)), (1470.0, dict(p_min=0.5)),
                     (3000.0, dict(p_min=0.5)), (1500.0, dict()), (200.0, dict(r_star=0.7, m_star=0.6, oversampling=2.0))]:
        okw = {("p_min_days" if k == "p_min" else k): v for k, v in kw.items()}
        assert g.gtls_period_grid_size(span, **kw) == oracle.period_grid(span, **okw).size
    for bad in [dict(span=0.0), dict(span=10.0, r_star=-1.0), dict(span=10.0, oversampling=0.0),
                dict(span=float("nan")), dict(span=1.0, p_min=0.5)]:
        with pytest.raises(g.GtlsError):
            g.gtls_period_grid_size(**bad)


def test_batch_workspace_bytes():
    co = np.array([0, 4000, 8200, 12000], dtype=np.int64)
    po = np.array([0, 10000, 20500, 30000], dtype=np.int64)
    a = g.gtls_batch_workspace_bytes(co, po, 25, period_tile=64)
    one = max(g.gtls_workspace_bytes(int(co[i + 1] - co[i]), int(po[i + 1] - po[i]), 25, period_tile=64) for i in range(3))
    lanes = int(os.environ.get("GTLS_BATCH_LANES", "1"))
    assert lanes * one <= a <= lanes * one + 4096    # every lane fits the largest curve
    assert g.gtls_batch_workspace_bytes(co[:2], po[:2], 25, period_tile=64) <= a
