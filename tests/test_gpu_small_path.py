"""GPU parity of the fused small-N path (gtls_opts.path = 1, csrc/small.cu: fold, sort, pad, scans and the
chi2 rings of one (curve, period) in one CTA's shared memory) against the CPU oracle, against the general
tiled path (path = 2), and through the survey-mode batch entry.  Bars as everywhere (north_star): best
(duration, start) indices bit-exact, chi2(P) within 1e-9 relative, SDE within 1e-6 absolute."""
import numpy as np
import pytest

import gtls_inputs as gi
import oracle
import paper_2607_00348_b200 as g

pytestmark = pytest.mark.gpu

CHI2_RTOL = 1e-9
SDE_ATOL = 1e-6


def _cuda():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    return torch


def _check(w, dt0, sde_kernel=31, label="", tmpl=None):
    tm = w.tmpl if tmpl is None else tmpl
    ora = oracle.search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, tm, dt0=dt0)
    res = g.gtls_search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, tm, dt0=dt0, sde_kernel=sde_kernel,
                        path=1, stats=True)
    assert res.stats["path"] == 1
    chi2, b = np.asarray(res.chi2), res.best()
    rel = np.abs(chi2 - ora.chi2) / np.maximum(np.abs(ora.chi2), 1e-300)
    assert rel.max() <= CHI2_RTOL, f"{label}: chi2 rel err {rel.max():.3e}"
    strict = ora.gap > 1e-12 * np.abs(ora.chi2)
    assert int((~strict).sum()) == 0, f"{label}: near-tie periods in the oracle"
    assert np.array_equal(b["dur_idx"], ora.best["dur_idx"]) and np.array_equal(b["start"], ora.best["start"]), label
    assert np.array_equal(b["t0"], ora.best["t0"]), label
    assert np.all(np.abs(b["depth"] - ora.best["depth"]) <= 1e-9 * np.abs(ora.best["depth"]) + 1e-18), label
    s = oracle.sde(ora.chi2, sde_kernel)
    assert np.abs(np.asarray(res.sde) - s.sde).max() <= SDE_ATOL, label
    assert res.summary["best_period_idx"] == s.best_period_idx and res.summary["sde_argmax"] == s.sde_argmax
    assert res.summary["windows_evaluated"] == ora.windows
    print(f"{label}: fused path, {w.n_per} periods, chi2 max rel err {rel.max():.2e}, min rel gap "
          f"{np.min(ora.gap / np.abs(ora.chi2)):.2e}")
    return res


def test_fused_c1_full():
    _cuda()
    w = gi.make_workload(1)
    res = _check(w, 0.05, sde_kernel=151, label="c1 fused")
    assert abs(res.summary["best_period"] - w.lc.meta["period"]) < 0.01


def test_fused_c2_full():
    _cuda()
    _check(gi.make_workload(2), 0.05, sde_kernel=151, label="c2 fused")


@pytest.mark.parametrize("cfg,every,dt0", [(1, 31, 0.0), (1, 13, 0.01), (2, 499, 0.0), (1, 7, 0.02), (1, 61, 0.1)])
def test_fused_other_skip_fractions(cfg, every, dt0):
    """Stride 1 (every duration becomes ceil(D / 24) window classes), small and large skip fractions."""
    _cuda()
    _check(gi.make_workload(cfg).subset(every), dt0, label=f"c{cfg}/{every} dt0={dt0}")


@pytest.mark.parametrize("curve", [0, 1, 2, 7])
def test_fused_survey_curves_c5(curve):
    _cuda()
    _check(gi.make_workload(5, curve=curve).subset(53), 0.05, label=f"c5.{curve} fused")


def test_fused_equals_general_path():
    """Same light curve through both paths: identical indices and t0, chi2 within rounding of each other
    (the two paths add the prefix sums in different orders)."""
    _cuda()
    w = gi.make_workload(2).subset(29)
    a = g.gtls_search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, w.tmpl, path=1, sde_kernel=31)
    b = g.gtls_search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, w.tmpl, path=2, sde_kernel=31, stats=True)
    assert b.stats["path"] == 2
    assert np.max(np.abs(np.asarray(a.chi2) / np.asarray(b.chi2) - 1)) <= 1e-12
    assert np.array_equal(a.best()[["dur_idx", "start", "t0"]], b.best()[["dur_idx", "start", "t0"]])
    assert a.summary["windows_evaluated"] == b.summary["windows_evaluated"]


def test_fused_ties_clusters_tiny_inputs_and_templates(tmpl512):
    _cuda()
    rng = np.random.default_rng(17)
    # tiny curves
    for n in (3, 4, 9, 40):
        t = np.sort(rng.uniform(0, 10, n)); y = 1 + rng.normal(0, 1e-3, n); dy = np.full(n, 1e-3)
        per = np.array([1.1, 2.7, 4.9]); qs = np.array([0.1, 0.3, 0.5])
        ora = oracle.search(t, y, dy, per, qs, tmpl512, dt0=0.0)
        res = g.gtls_search(t, y, dy, per, qs, tmpl512, dt0=0.0, sde_kernel=3, path=1)
        assert np.allclose(res.chi2, ora.chi2, rtol=CHI2_RTOL, atol=0), n
        b = res.best()
        assert np.array_equal(b["dur_idx"], ora.best["dur_idx"]) and np.array_equal(b["start"], ora.best["start"])
        assert np.array_equal(b["t0"], ora.best["t0"])
    # phases that cluster into one sort bin, exact phase ties (stable by index), equal 32-bit keys
    n = 3000
    t = np.arange(n) * 0.5 + rng.uniform(0, 1e-4, n)
    t[100:200] = np.arange(100, 200) * 0.5                      # exact multiples: phase 0 for P = 0.5
    y = 1 + rng.normal(0, 1e-3, n); dy = np.full(n, 1e-3)
    per = np.array([0.5, 0.37, 1.0, 0.25]); qs = np.array([0.01, 0.05, 0.1])
    ora = oracle.search(t, y, dy, per, qs, tmpl512, dt0=0.05)
    res = g.gtls_search(t, y, dy, per, qs, tmpl512, dt0=0.05, sde_kernel=3, path=1)
    assert np.allclose(res.chi2, ora.chi2, rtol=CHI2_RTOL, atol=0)
    b = res.best()
    assert np.array_equal(b["dur_idx"], ora.best["dur_idx"]) and np.array_equal(b["start"], ora.best["start"])
    assert np.array_equal(b["t0"], ora.best["t0"])
    # templates the shared-memory cache / the TMA bulk copy cannot take
    w = gi.make_workload(1).subset(97)
    for n_tmpl in (2, 7, 513, 2048):
        tm = gi.transit_template(n_tmpl) if n_tmpl > 2 else np.array([1.0, 1.0])
        _check(w, 0.05, sde_kernel=5, label=f"fused n_tmpl={n_tmpl}", tmpl=tm)
    # flat curve (reading G22) and brightening-only curve (G7)
    t = np.linspace(0, 10, 40)
    res = g.gtls_search(t, np.ones(40), np.full(40, 1e-3), np.array([1.1, 2.2]), np.array([0.1, 0.2]), tmpl512, path=1)
    assert res.code == -6 and np.all(res.chi2 == 0) and np.all(res.sde == 0)
    assert np.all(res.best()["dur_idx"] == 0) and np.all(res.best()["start"] == 0)
    y = 1.0 + np.abs(rng.normal(0, 1e-3, 40))
    res = g.gtls_search(t, y, np.full(40, 1e-3), np.array([1.7]), np.array([0.1, 0.3]), tmpl512, dt0=0.0, path=1)
    assert res.chi2[0] == res.summary["chi2_null"] and res.best()["depth"][0] == 0.0


def test_fused_path_limits():
    """path = 1 is refused (GTLS_EUNSUPPORTED) where the fused kernel does not apply; path = 0 then takes
    the general path by itself."""
    _cuda()
    w = gi.make_workload(1, hetero=True).subset(97)              # per-point errors
    with pytest.raises(g.GtlsError) as e:
        g.gtls_search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, w.tmpl, path=1)
    assert e.value.code == -7
    assert g.gtls_search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, w.tmpl, stats=True).stats["path"] == 2
    w = gi.make_workload(2).subset(499)
    with pytest.raises(g.GtlsError) as e:                        # class strides above 31 columns (dt0 = 0.1, D = 628)
        g.gtls_search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, w.tmpl, dt0=0.1, path=1)
    assert e.value.code == -7
    w3 = gi.make_workload(3).subset(50000)                       # 65 000 points do not fit a CTA
    with pytest.raises(g.GtlsError) as e:
        g.gtls_search(w3.lc.t, w3.lc.y, w3.lc.dy, w3.periods, w3.durations, w3.tmpl, path=1)
    assert e.value.code == -7


def test_fused_batch_is_one_launch_and_matches_oracle():
    """gtls_search_batch on uniform-dy curves: one fused kernel over every (curve, period); results equal
    single calls bit for bit and the oracle to the usual bars; per-curve summaries and statuses."""
    torch = _cuda()
    ws = [gi.make_workload(5, curve=c).subset(61) for c in range(9)]
    cat = lambda xs, ax=0: np.ascontiguousarray(np.concatenate(xs, axis=ax))
    t, y, dy = (cat([getattr(w.lc, k) for w in ws]) for k in ("t", "y", "dy"))
    per, dur = cat([w.periods for w in ws]), cat([w.durations for w in ws])
    co = np.concatenate([[0], np.cumsum([w.lc.n for w in ws])]).astype(np.int64)
    po = np.concatenate([[0], np.cumsum([w.n_per for w in ws])]).astype(np.int64)
    tm = ws[0].tmpl
    f = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    res = g.gtls_search_batch(f(t), f(y), f(dy), co, f(per), po, f(dur), f(tm), dt0=0.05, sde_kernel=31, path=1)
    chi2, sde, best = res.chi2.cpu().numpy(), res.sde.cpu().numpy(), res.best()
    assert np.all(res.status == 0)
    for c, w in enumerate(ws):
        sl = slice(po[c], po[c + 1])
        one = g.gtls_search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, tm, dt0=0.05, sde_kernel=31, path=1)
        assert np.array_equal(chi2[sl], one.chi2) and np.array_equal(sde[sl], one.sde)
        assert np.array_equal(best[sl], one.best())
        assert res.summaries[c] == one.summary
        ora = oracle.search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, tm, dt0=0.05)
        assert np.max(np.abs(chi2[sl] / ora.chi2 - 1.0)) <= CHI2_RTOL
        assert np.array_equal(best[sl]["dur_idx"], ora.best["dur_idx"]) and np.array_equal(best[sl]["start"], ora.best["start"])
        s = oracle.sde(ora.chi2, 31)
        assert np.abs(sde[sl] - s.sde).max() <= SDE_ATOL
        assert res.summaries[c]["best_period_idx"] == s.best_period_idx
        assert res.summaries[c]["windows_evaluated"] == ora.windows
