"""GPU parity of the device-built trial grids (paper section 2.2) and of the survey-mode batch entry
(BASELINE.json config 5) against the CPU oracle and against single gtls_search calls."""
import numpy as np
import pytest

import gtls_inputs as gi
import oracle
import paper_2607_00348_b200 as g

pytestmark = pytest.mark.gpu

# period grid: the kernel's cube and divisions are exact IEEE operations, only the host-side constants A, C
# (pow against the oracle's cbrt) may differ by an ulp, which the cube triples
GRID_RTOL = 1e-14
# duration grid: device pow / log / exp are accurate to 1-2 ulp each; ln q ~ -7 amplifies their absolute
# error into ~1e-15 relative on q
DUR_RTOL = 1e-13


def _cuda():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    return torch


@pytest.mark.parametrize("span,kw", [(30.0, dict(p_min=0.5)), (90.0, dict(p_min=0.5)), (1500.0, dict()),
                                     (3000.0, dict(p_min=0.5)), (90.0, dict(p_min=0.5, oversampling=5.0)),
                                     (400.0, dict(r_star=0.6, m_star=0.55))])
def test_period_grid_matches_oracle(span, kw):
    torch = _cuda()
    okw = {("p_min_days" if k == "p_min" else k): v for k, v in kw.items()}
    ref = oracle.period_grid(span, **okw)
    host = g.gtls_period_grid(span, **kw)                                   # host output
    assert host.shape == ref.shape
    assert np.max(np.abs(host / ref - 1.0)) <= GRID_RTOL
    dev = g.gtls_period_grid(span, device=torch.device("cuda:0"), **kw)     # device output
    assert np.array_equal(dev.cpu().numpy(), host)
    assert abs(host[0] - span / 2) <= 1e-9 * span                           # Eq. 1
    assert np.all(np.diff(host) < 0)


def test_period_grid_size_matches_survey_table_and_paper():
    _cuda()
    assert g.gtls_period_grid(1500.0).size == 191748                        # N ~ 190 000
    for cfg, span in ((1, 30.0), (2, 90.0)):                                # SURVEY.md section 8 workload table
        assert g.gtls_period_grid(span, p_min=0.5).size == gi.make_workload(cfg).n_per


@pytest.mark.parametrize("n_dur", [1, 2, 25, 30])
def test_duration_grid_matches_oracle(n_dur):
    torch = _cuda()
    p = oracle.period_grid(1470.0, p_min_days=0.5)[::37]
    ref = oracle.duration_grid(p, n_dur)
    host = g.gtls_duration_grid(p, n_dur)
    assert host.shape == ref.shape
    assert np.max(np.abs(host / ref - 1.0)) <= DUR_RTOL
    dev = g.gtls_duration_grid(torch.from_numpy(p).cuda(), n_dur)
    assert np.array_equal(dev.cpu().numpy(), host)
    assert host.max() <= 0.15
    tls = g.gtls_duration_grid(p, n_dur, 41.39, 546.94, 0.112)              # TLS constants
    assert np.max(np.abs(tls / oracle.duration_grid(p, n_dur, 41.39, 546.94, 0.112) - 1.0)) <= DUR_RTOL


def test_grid_errors():
    _cuda()
    with pytest.raises(g.GtlsError):
        g.gtls_period_grid(-1.0)
    with pytest.raises(g.GtlsError):
        g.gtls_period_grid(1.0, p_min=0.5)                                  # f_max <= f_min
    with pytest.raises(g.GtlsError):
        g.gtls_duration_grid(np.array([1.0, -2.0]), 5)                      # GTLS_EGRID
    with pytest.raises(g.GtlsError):
        g.gtls_duration_grid(np.array([1.0]), 5, 10.0, 5.0)                 # k_max < k_min


def test_search_on_device_built_grids():
    """The whole front end on the device: grids from gtls_period_grid / gtls_duration_grid feed gtls_search;
    the oracle searches its own grids; spectra agree (D = floor(q n) is the same for both grids here)."""
    torch = _cuda()
    w = gi.make_workload(1)
    dev = torch.device("cuda:0")
    per = g.gtls_period_grid(30.0, p_min=0.5, device=dev)[::61].contiguous()
    dur = g.gtls_duration_grid(per, 20)
    tt = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    res = g.gtls_search(tt(w.lc.t), tt(w.lc.y), tt(w.lc.dy), per, dur, tt(w.tmpl), dt0=0.05, sde_kernel=5)
    op = np.ascontiguousarray(oracle.period_grid(30.0, p_min_days=0.5)[::61])
    oq = oracle.duration_grid(op, 20)
    n = w.lc.n
    assert np.array_equal(np.floor(oq * n), np.floor(dur.cpu().numpy() * n))
    ora = oracle.search(w.lc.t, w.lc.y, w.lc.dy, op, oq, w.tmpl, dt0=0.05)
    chi2 = res.chi2.cpu().numpy()
    assert np.max(np.abs(chi2 / ora.chi2 - 1.0)) <= 1e-9
    best = res.best()
    assert np.array_equal(best["dur_idx"], ora.best["dur_idx"]) and np.array_equal(best["start"], ora.best["start"])


def _batch_inputs(curves, every):
    ws = [gi.make_workload(5, curve=c).subset(every, offset=c % every) for c in curves]
    t = np.concatenate([w.lc.t for w in ws]); y = np.concatenate([w.lc.y for w in ws])
    dy = np.concatenate([w.lc.dy for w in ws])
    per = np.concatenate([w.periods for w in ws]); dur = np.concatenate([w.durations for w in ws], axis=0)
    co = np.concatenate([[0], np.cumsum([w.lc.n for w in ws])]).astype(np.int64)
    po = np.concatenate([[0], np.cumsum([w.n_per for w in ws])]).astype(np.int64)
    return ws, t, y, dy, co, per, po, dur


@pytest.mark.parametrize("device_mode", [False, True])
def test_search_batch_equals_single_calls_and_oracle(device_mode):
    torch = _cuda()
    curves = [0, 1, 2, 3, 4, 5, 6]                       # more curves than lanes, ragged n and n_per
    ws, t, y, dy, co, per, po, dur = _batch_inputs(curves, 97)
    tm = ws[0].tmpl
    if device_mode:
        f = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
        res = g.gtls_search_batch(f(t), f(y), f(dy), co, f(per), po, f(dur), f(tm), dt0=0.05, sde_kernel=31)
        chi2, sde, sde_raw = res.chi2.cpu().numpy(), res.sde.cpu().numpy(), res.sde_raw.cpu().numpy()
    else:
        res = g.gtls_search_batch(t, y, dy, co, per, po, dur, tm, dt0=0.05, sde_kernel=31)
        chi2, sde, sde_raw = res.chi2, res.sde, res.sde_raw
    best = res.best()
    assert np.all(res.status == 0)
    for c, w in enumerate(ws):
        sl = slice(po[c], po[c + 1])
        one = g.gtls_search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, tm, dt0=0.05, sde_kernel=31)
        assert np.array_equal(chi2[sl], one.chi2)                          # same kernels: bit for bit
        assert np.array_equal(sde[sl], one.sde) and np.array_equal(sde_raw[sl], one.sde_raw)
        assert np.array_equal(best[sl], one.best())
        assert res.summaries[c] == one.summary
        ora = oracle.search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, tm, dt0=0.05)
        assert np.max(np.abs(chi2[sl] / ora.chi2 - 1.0)) <= 1e-9
        strict = ora.gap > 1e-12 * np.abs(ora.chi2)
        mism = (best[sl]["dur_idx"] != ora.best["dur_idx"]) | (best[sl]["start"] != ora.best["start"])
        assert not np.any(mism & strict)
        s = oracle.sde(ora.chi2, 31)
        assert np.abs(sde[sl] - s.sde).max() <= 1e-6
        assert res.summaries[c]["best_period_idx"] == s.best_period_idx


def test_search_batch_shared_durations_workspace_and_status():
    """Shared duration grid, caller-owned scratch, a flat curve (degenerate) and a curve with a bad dy:
    the other curves are still searched and the first hard error is returned."""
    torch = _cuda()
    ws, t, y, dy, co, per, po, _ = _batch_inputs([0, 1, 2], 211)
    q = np.geomspace(0.004, 0.08, 9)
    tm = ws[0].tmpl
    f = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    nbytes = g.gtls_batch_workspace_bytes(co, po, 9)
    assert nbytes > 0
    wsp = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    res = g.gtls_search_batch(f(t), f(y), f(dy), co, f(per), po, f(q), f(tm), sde_kernel=0, workspace=wsp)
    for c, w in enumerate(ws):
        one = g.gtls_search(w.lc.t, w.lc.y, w.lc.dy, w.periods, q, tm, sde_kernel=0)
        assert np.array_equal(res.chi2.cpu().numpy()[po[c]:po[c + 1]], one.chi2)
    with pytest.raises(g.GtlsError):                                       # scratch too small
        g.gtls_search_batch(f(t), f(y), f(dy), co, f(per), po, f(q), f(tm), workspace=wsp[:4096])
    y2 = y.copy(); y2[co[1]:co[2]] = 1.0                                    # curve 1 flat: chi2 = 0 everywhere
    res = g.gtls_search_batch(t, y2, dy, co, per, po, q, tm, sde_kernel=0)
    assert list(res.status) == [0, g.GTLS_EDEGENERATE, 0]
    assert np.all(res.chi2[po[1]:po[2]] == 0.0)
    dy2 = dy.copy(); dy2[co[2] + 5] = -1.0                                  # curve 2 invalid
    import ctypes as C
    lib = g.load_library()
    o = g.GtlsOpts(); lib.gtls_opts_default(C.byref(o)); o.sde_kernel = 0
    chi2 = np.full(po[-1], -7.0); status = np.zeros(3, dtype=np.int32)
    rc = lib.gtls_search_batch(3, t.ctypes.data, y.ctypes.data, dy2.ctypes.data, co.ctypes.data, per.ctypes.data,
                               po.ctypes.data, q.ctypes.data, 9, tm.ctypes.data, tm.size, C.byref(o),
                               chi2.ctypes.data, None, None, None, None, status.ctypes.data)
    assert rc == -2 and list(status) == [0, 0, -2]                           # GTLS_ENONFINITE


def test_block_pool_reuse_and_release():
    """Host-buffer calls keep their device blocks between calls: results do not depend on whether a block is
    fresh or reused (also by a call of another size), and gtls_release_cache gives the memory back."""
    torch = _cuda()
    g.gtls_release_cache()
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    w = gi.make_workload(2).subset(211)
    a = g.gtls_search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, w.tmpl, sde_kernel=5)      # fresh blocks
    held = free0 - torch.cuda.mem_get_info()[0]
    assert held > 0                                                                                # pooled
    w1 = gi.make_workload(1).subset(61)
    c = g.gtls_search(w1.lc.t, w1.lc.y, w1.lc.dy, w1.periods, w1.durations, w1.tmpl, sde_kernel=5)  # smaller: reuses
    b = g.gtls_search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, w.tmpl, sde_kernel=5)      # reused blocks
    assert np.array_equal(a.chi2, b.chi2) and np.array_equal(a.best(), b.best()) and np.array_equal(a.sde, b.sde)
    ora = oracle.search(w1.lc.t, w1.lc.y, w1.lc.dy, w1.periods, w1.durations, w1.tmpl, dt0=0.05)
    assert np.max(np.abs(c.chi2 / ora.chi2 - 1.0)) <= 1e-9
    with pytest.raises(g.GtlsError):                                                               # error path returns its blocks too
        bad = w.lc.dy.copy(); bad[3] = 0.0
        g.gtls_search(w.lc.t, w.lc.y, bad, w.periods, w.durations, w.tmpl)
    assert torch.cuda.mem_get_info()[0] >= free0 - 2 * held - (64 << 20)                           # bounded, no growth per call
    g.gtls_release_cache()
    assert torch.cuda.mem_get_info()[0] >= free0 - (8 << 20)


def test_search_batch_concurrent_lanes_subprocess():
    """GTLS_BATCH_LANES is read once per process: three concurrent lanes (host threads, one stream and one
    scratch slice each) in a child process, results bit-identical to single calls."""
    _cuda()
    import os, subprocess, sys
    code = r'''
import numpy as np, gtls_inputs as gi, paper_2607_00348_b200 as g
ws = [gi.make_workload(5, curve=c).subset(131, offset=c) for c in range(7)]
cat = lambda xs: np.ascontiguousarray(np.concatenate(xs, axis=0))
co = np.concatenate([[0], np.cumsum([w.lc.n for w in ws])]).astype(np.int64)
po = np.concatenate([[0], np.cumsum([w.n_per for w in ws])]).astype(np.int64)
res = g.gtls_search_batch(cat([w.lc.t for w in ws]), cat([w.lc.y for w in ws]), cat([w.lc.dy for w in ws]), co,
                          cat([w.periods for w in ws]), po, cat([w.durations for w in ws]), ws[0].tmpl, sde_kernel=21)
assert g.gtls_batch_workspace_bytes(co, po, 25) >= 3 * max(g.gtls_workspace_bytes(w.lc.n, w.n_per, 25) for w in ws)
for c, w in enumerate(ws):
    one = g.gtls_search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, w.tmpl, sde_kernel=21)
    sl = slice(po[c], po[c + 1])
    assert np.array_equal(res.chi2[sl], one.chi2) and np.array_equal(res.sde[sl], one.sde)
    assert np.array_equal(res.best()[sl], one.best()) and res.summaries[c] == one.summary
print("lanes ok")
'''
    env = dict(os.environ, GTLS_BATCH_LANES="3")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, "-c", code], cwd=root, env=env, capture_output=True, text=True, timeout=600)
    assert out.returncode == 0 and "lanes ok" in out.stdout, out.stderr[-2000:]
