"""gtls_search_static: the allocation-free entry point (all scratch in one static device array of
gtls_static_scratch_bytes(), csrc/api_static.cu) against the existing fused path (gtls_search, path = 1) and
the CPU oracle, on two calls in a row that share the array.  Collected last on purpose (the file name): the
suite runs with pytest -x."""
import numpy as np
import pytest

import gtls_inputs as gi
import oracle
import paper_2607_00348_b200 as g

pytestmark = pytest.mark.gpu

CHI2_RTOL = 1e-9
SDE_ATOL = 1e-6


def _dev(torch, w):
    f = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return [f(x) for x in (w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, w.tmpl)]


def _compare(torch, w, res, label):
    ref = g.gtls_search(*_dev(torch, w), dt0=0.05, sde_kernel=31, path=1)          # the existing path
    chi2, rchi2 = res.chi2.cpu().numpy(), ref.chi2.cpu().numpy()
    assert np.max(np.abs(chi2 - rchi2) / np.abs(rchi2)) <= CHI2_RTOL, label
    b, rb = res.best(), ref.best()
    assert np.array_equal(b["dur_idx"], rb["dur_idx"]) and np.array_equal(b["start"], rb["start"]), label
    assert np.array_equal(b["t0"], rb["t0"]), label
    assert np.abs(res.sde.cpu().numpy() - ref.sde.cpu().numpy()).max() <= SDE_ATOL, label
    assert np.abs(res.sde_raw.cpu().numpy() - ref.sde_raw.cpu().numpy()).max() <= SDE_ATOL, label
    for k in ("best_period_idx", "best_dur_idx", "best_start", "sde_argmax", "windows_evaluated"):
        assert res.summary[k] == ref.summary[k], (label, k)
    assert abs(res.summary["chi2_min"] / ref.summary["chi2_min"] - 1) <= CHI2_RTOL
    assert abs(res.summary["sde_max"] - ref.summary["sde_max"]) <= SDE_ATOL
    # and the oracle, to the bars of the parity tests
    ora = oracle.search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, w.tmpl, dt0=0.05)
    assert np.max(np.abs(chi2 - ora.chi2) / ora.chi2) <= CHI2_RTOL, label
    assert np.array_equal(b["dur_idx"], ora.best["dur_idx"]) and np.array_equal(b["start"], ora.best["start"]), label
    assert np.abs(res.sde.cpu().numpy() - oracle.sde(ora.chi2, 31).sde).max() <= SDE_ATOL, label


def test_static_scratch_entry_point_two_calls_in_a_row():
    import torch
    assert torch.cuda.is_available(), "this test needs a CUDA device"
    assert 0 < g.gtls_static_scratch_bytes() <= 1 << 20                             # a modest, fixed size
    w1 = gi.make_workload(2).subset(97)            # 4 188 points, 109 periods x 25 durations
    w2 = gi.make_workload(1).subset(13)            # another curve, another size: the array holds w1's leftovers
    # outputs are the caller's: allocate them (and everything else) BEFORE the calls under test
    d1, d2 = _dev(torch, w1), _dev(torch, w2)
    mk = lambda n: (torch.empty(n, dtype=torch.float64, device="cuda"), torch.empty((n, 24), dtype=torch.uint8, device="cuda"),
                    torch.empty(n, dtype=torch.float64, device="cuda"), torch.empty(n, dtype=torch.float64, device="cuda"))
    o1, o2, o3 = mk(w1.n_per), mk(w2.n_per), mk(w1.n_per)
    # one untimed call first: the driver loads a kernel's code into device memory at its first launch (lazy
    # module loading), which is the library being loaded, not the entry point allocating
    g.gtls_search_static(*d2, dt0=0.05, sde_kernel=31, out=o2)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    r1 = g.gtls_search_static(*d1, dt0=0.05, sde_kernel=31, out=o1)
    r2 = g.gtls_search_static(*d2, dt0=0.05, sde_kernel=31, out=o2)                 # second call, same scratch
    r3 = g.gtls_search_static(*d1, dt0=0.05, sde_kernel=31, out=o3)                 # and the first problem again
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0, "the calls changed the device's free memory"
    _compare(torch, w1, r1, "first call")
    _compare(torch, w2, r2, "second call")
    assert torch.equal(r3.chi2, r1.chi2) and torch.equal(r3.sde, r1.sde) and np.array_equal(r3.best(), r1.best())


def test_static_scratch_entry_point_rejects_what_does_not_fit():
    import torch
    assert torch.cuda.is_available(), "this test needs a CUDA device"
    f = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    rng = np.random.default_rng(5)
    n = 8193                                                                         # one point beyond the maximum
    t = np.sort(rng.uniform(0, 90, n)); y = 1 + rng.normal(0, 1e-3, n); dy = np.full(n, 1e-3)
    tm = gi.transit_template(512)
    with pytest.raises(g.GtlsError) as e:
        g.gtls_search_static(f(t), f(y), f(dy), f(np.array([1.3, 2.9])), f(np.array([0.01, 0.02])), f(tm))
    assert e.value.code == -7 and "8192" in str(e.value)
    w = gi.make_workload(1, hetero=True).subset(97)                                  # per-point errors
    with pytest.raises(g.GtlsError) as e:
        g.gtls_search_static(*_dev(torch, w))
    assert e.value.code == -7 and "uniform" in str(e.value)
    w = gi.make_workload(1).subset(97)                                               # and a call that fits still works
    r = g.gtls_search_static(*_dev(torch, w), sde_kernel=31)
    ref = g.gtls_search(*_dev(torch, w), sde_kernel=31, path=1)
    assert torch.equal(r.chi2, ref.chi2) and np.array_equal(r.best(), ref.best())
