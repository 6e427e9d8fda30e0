"""Oracle pins for the per-step functions: fold (P4), sort (P5), template (P8), stride (P11),
SDE (P9) and the median detrend (P10).  None of these checks retypes the oracle's formula:
they use closed forms, library routines and the paper's printed example."""
import json
import os

import numpy as np
import pytest
from scipy.ndimage import median_filter

import oracle

PINS = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_pins.json")))


# ---------------------------------------------------------------- P4 fold (Eq. 10)
def test_fold_range_and_exact_multiples():
    rng = np.random.default_rng(1)
    t = rng.uniform(0, 3000, 5000)
    for period in (0.5, 3.7, 213.0, 1499.9):
        p = oracle.fold(t, period)
        assert np.all(p >= 0.0) and np.all(p <= 1.0)
        # the phase times P lands back on t modulo P
        k = np.round((t - p * period) / period)
        assert np.allclose(k * period + p * period, t, rtol=0, atol=1e-9)
    period = 2.5
    t = np.arange(40) * period                       # t = k P exactly => p = 0
    assert np.all(oracle.fold(t, period) == 0.0)
    # binary-exact case: quarter steps of P=2 give phases {0, .25, .5, .75} exactly
    t = np.arange(64) / 2.0
    assert np.array_equal(oracle.fold(t, 2.0), (np.arange(64) % 4) / 4.0)


def test_fold_negative_times_stay_in_unit_interval():
    p = oracle.fold(np.array([-1e-18, -0.25, -3.0]), 1.0)
    assert p[0] == 1.0 and p[1] == 0.75 and p[2] == 0.0   # reading G1: phase may round to 1.0


# ---------------------------------------------------------------- P5 sort
def test_sort_matches_numpy_stable_argsort():
    rng = np.random.default_rng(2)
    t = np.sort(rng.uniform(0, 90, 3000))
    periods = np.array([0.5, 1.2345, 11.2, 44.9])
    phase, perm = oracle.fold_sort(t, periods)
    for k, P in enumerate(periods):
        assert np.array_equal(perm[k], np.argsort(phase[k], kind="stable"))
        assert sorted(perm[k]) == list(range(t.size))


def test_sort_ties_keep_original_index_order():
    t = np.arange(64) / 2.0                          # P=2 => phases in {0,1/4,1/2,3/4}
    _, perm = oracle.fold_sort(t, [2.0])
    expect = np.concatenate([np.arange(r, 64, 4) for r in range(4)])
    assert np.array_equal(perm[0], expect)
    t = np.arange(50) * 3.0                          # all phases equal => identity
    _, perm = oracle.fold_sort(t, [3.0])
    assert np.array_equal(perm[0], np.arange(50))


# ---------------------------------------------------------------- P8 template resampling
def test_template_constant_and_linear_are_exact():
    for d in (1, 2, 7, 100, 2523):
        g, gbar = oracle.resample_template(np.full(33, 0.7), d)
        assert np.all(g == 0.7) and abs(gbar - 0.7) < 1e-13
        g, gbar = oracle.resample_template(np.linspace(0.0, 1.0, 129), d)
        assert np.allclose(g, (np.arange(d) + 0.5) / d, rtol=0, atol=2e-15)
        assert abs(gbar - 0.5) < 1e-13


def test_template_symmetry_and_integral_limit(tmpl512):
    for d in (5, 44, 627):
        g, gbar = oracle.resample_template(tmpl512, d)
        assert np.allclose(g, g[::-1], atol=1e-12)
        assert abs(gbar - g.mean()) < 1e-15
    integral = np.trapezoid(tmpl512, np.linspace(0, 1, 512))
    errs = [abs(oracle.resample_template(tmpl512, d)[1] - integral) for d in (10, 100, 1000, 10000)]
    assert errs[0] > errs[1] > errs[2] and errs[3] < 1e-5


def test_template_node_hits():
    # D = n_tmpl-1 cells: centres fall exactly half-way between nodes
    tm = np.array([0.0, 1.0, 4.0, 9.0, 16.0])
    g, _ = oracle.resample_template(tm, 4)
    assert np.allclose(g, [0.5, 2.5, 6.5, 12.5])


# ---------------------------------------------------------------- P11 stride (Eq. 18)
def test_stride_paper_example_and_floor():
    ex = PINS["skip_example"]
    assert oracle.stride(ex["n_it"], ex["dt0"]) == ex["n_skip"]
    assert oracle.stride(2000, 0.0) == 1 and oracle.stride(5, 0.05) == 1
    assert oracle.stride(39, 0.05) == 1 and oracle.stride(40, 0.05) == 2
    assert oracle.stride(19837, 0.05) == 991


def test_points_in_duration_clamps():
    assert oracle.points_in_duration(0.15, 4188) == 628
    assert oracle.points_in_duration(1e-9, 4188) == 1
    assert oracle.points_in_duration(0.9999, 100) == 99 and oracle.points_in_duration(5.0, 100) == 99


# ---------------------------------------------------------------- P9 / P10 SDE (Eq. 17)
def test_sde_closed_forms():
    rng = np.random.default_rng(3)
    chi2 = 1000.0 + rng.normal(0, 3, 4000) - 0.01 * np.arange(4000)
    chi2[1234] = 900.0
    s = oracle.sde(chi2, 0)
    assert not s.degenerate and s.best_period_idx == 1234
    assert np.allclose(s.sr, 900.0 / chi2, rtol=1e-15)        # reading G15: SR <= 1
    assert abs(s.sde_raw.mean()) < 1e-10 and abs(s.sde_raw.std() - 1.0) < 1e-12
    assert abs(s.sde_raw.max() - (1 - s.sr.mean()) / s.sr.std()) < 1e-10
    assert int(np.argmax(s.sde_raw)) == 1234
    assert np.array_equal(s.sde, s.sde_raw)                   # kernel 0 => no detrend


@pytest.mark.parametrize("kernel,n", [(151, 4000), (31, 200), (151, 60), (3, 10)])
def test_sde_median_detrend_matches_scipy(kernel, n):
    rng = np.random.default_rng(kernel + n)
    chi2 = 500.0 + np.cumsum(rng.normal(0, 0.2, n)) + rng.normal(0, 1, n)
    s = oracle.sde(chi2, kernel)
    expect = s.sde_raw - median_filter(s.sde_raw, size=kernel, mode="nearest")
    assert np.allclose(s.sde, expect, rtol=0, atol=1e-13)
    assert s.sde_argmax == int(np.argmax(expect))


def test_sde_degenerate():
    s = oracle.sde(np.zeros(10), 5)
    assert s.degenerate and np.all(s.sde == 0)
    s = oracle.sde(np.full(10, 3.0), 5)
    assert s.degenerate and np.all(s.sde_raw == 0)


def test_two_stage_refinement_properties(tmpl512):
    """Section 2.5 on the oracle: n_refine >= n_per equals the stride-1 search;
    refinement never raises chi2 and leaves unselected periods untouched; selection = highest SDE."""
    import gtls_inputs as gi
    w = gi.make_workload(1).subset(127)
    full = oracle.search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, tmpl512, dt0=0.0)
    coarse = oracle.search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, tmpl512, dt0=0.1)
    ts_all = oracle.search_two_stage(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, tmpl512, dt0=0.1,
                                     n_refine=10 ** 6, sde_kernel=5)
    assert np.array_equal(ts_all.chi2, full.chi2) and np.array_equal(ts_all.best, full.best)
    ts = oracle.search_two_stage(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, tmpl512, dt0=0.1,
                                 n_refine=5, sde_kernel=5)
    assert ts.refined.size == 5
    assert np.all(ts.chi2 <= coarse.chi2)
    rest = np.setdiff1d(np.arange(w.n_per), ts.refined)
    assert np.array_equal(ts.chi2[rest], coarse.chi2[rest])
    assert np.array_equal(ts.chi2[ts.refined], full.chi2[ts.refined])
    assert ts.coarse_sde[ts.refined].min() >= np.delete(ts.coarse_sde, ts.refined).max()
