"""Oracle pins for the chi^2 search: P1 brute force against the literal padded form of the
paper (Fig. 3, Eq. 11, 15, 16), P2 closed-form box case, P3 injected-transit recovery,
P7 invariants, P11 stride monotonicity, P13 noise-free folded-domain construction, P14 top-K.
The numpy code here is written from the paper's padded formulation / closed forms, not from
the oracle's circular direct sums."""
import numpy as np
import pytest

import gtls_inputs as gi
import oracle


def _tiny_curve(seed, n=48, hetero=True):
    rng = np.random.default_rng(seed)
    t = np.sort(rng.uniform(0.0, 20.0, n))
    y = 1.0 + rng.normal(0, 1e-3, n)
    dy = 1e-3 * (rng.uniform(0.5, 2.0, n) if hetero else np.ones(n))
    return t, y, dy


def _padded_literal(t, y, dy, period, d, d_m, g, gbar):
    """Fig. 3 + Eq. 11, 15, 16 taken literally on the padded folded curve (reading G4):
    returns chi2[s] for every start s in [0, N)."""
    n = t.size
    phase = t / period - np.floor(t / period)
    sig = np.argsort(phase, kind="stable")
    f = np.concatenate([y[sig], y[sig][:d_m]])            # pad: first D_m points appended
    e = np.concatenate([dy[sig], dy[sig][:d_m]])
    n_p = n + d_m
    edge = np.sum(((1.0 - f[n:]) / e[n:]) ** 2)           # Eq. 11 over the pad region
    out = np.empty(n)
    depth = np.empty(n)
    for s in range(n):
        ds, de = s, s + d                                 # window [ds, de)
        w = 1.0 / e[ds:de] ** 2
        fbar = np.sum(w * f[ds:de]) / np.sum(w)
        a = max(1.0 - fbar, 0.0) / gbar                   # Eq. 12-13 (readings G5-G7)
        chi_a = np.sum(((f[:ds] - 1.0) / e[:ds]) ** 2)    # Eq. 15, before
        chi_b = np.sum(((f[de:n_p] - 1.0) / e[de:n_p]) ** 2)   # Eq. 15, after
        f_ideal = 1.0 - a * g
        chi_in = np.sum(((f[ds:de] - f_ideal) / e[ds:de]) ** 2)  # Eq. 16
        out[s] = chi_a + chi_b - edge + chi_in
        depth[s] = a
    return out, depth, sig


# ------------------------------------------------------------------------------ P1
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_brute_force_padded_literal_equals_oracle(seed, tmpl512):
    t, y, dy = _tiny_curve(seed)
    n = t.size
    periods = np.array([1.7, 3.3, 9.1])
    qs = np.array([2.5 / n, 5.2 / n, 9.9 / n, 14.0 / n])     # D = 2, 5, 9, 14
    d_m = 14
    res = oracle.search(t, y, dy, periods, qs, tmpl512, dt0=0.0)
    for ip, period in enumerate(periods):
        best = (np.inf, -1, -1)
        for jd, q in enumerate(qs):
            d = oracle.points_in_duration(q, n)
            g, gbar = oracle.resample_template(tmpl512, d)
            lit, depth, sig = _padded_literal(t, y, dy, period, d, d_m, g, gbar)
            st, dep, c_out, c_in = oracle.window_chi2_literal(t, y, dy, period, q, tmpl512, 0.0)
            assert np.array_equal(st, np.arange(n))
            assert np.allclose(c_out + c_in, lit, rtol=1e-13, atol=0)     # circular == padded
            assert np.allclose(dep, depth, rtol=1e-10, atol=1e-15)   # 1 - fbar cancels ~1e-16 abs
            s = int(np.argmin(lit))
            if lit[s] < best[0]:
                best = (lit[s], jd, s)
        assert abs(res.chi2[ip] / best[0] - 1.0) < 1e-13
        assert (res.best["dur_idx"][ip], res.best["start"][ip]) == (best[1], best[2])


def test_search_chi2_equals_literal_minimum_with_stride(tmpl512):
    t, y, dy = _tiny_curve(7, n=64)
    q = 41.0 / 64
    st, dep, c_out, c_in = oracle.window_chi2_literal(t, y, dy, 2.9, q, tmpl512, 0.1)
    assert np.array_equal(st, np.arange(0, 64, 4))                 # D=41, stride floor(4.1)=4
    res = oracle.search(t, y, dy, [2.9], [q], tmpl512, dt0=0.1)
    k = int(np.argmin(c_out + c_in))
    assert abs(res.chi2[0] / (c_out + c_in)[k] - 1.0) < 1e-13
    assert res.best["start"][0] == st[k] and abs(res.best["depth"][0] - dep[k]) < 1e-15
    assert res.windows == 16


# ------------------------------------------------------------------------------ P2 / P6
@pytest.mark.parametrize("hetero", [False, True])
def test_box_template_reduces_to_bls_closed_form(hetero):
    t, y, dy = _tiny_curve(11, n=60, hetero=hetero)
    n = t.size
    box = np.ones(16)
    periods = np.array([2.2, 5.7])
    qs = np.array([3.5 / n, 8.5 / n])
    res = oracle.search(t, y, dy, periods, qs, box, dt0=0.0)
    w = 1.0 / dy ** 2
    r = 1.0 - y
    chi0 = np.sum(w * r * r)
    assert abs(res.chi2_null / chi0 - 1) < 1e-14
    for ip, period in enumerate(periods):
        sig = np.argsort(t / period - np.floor(t / period), kind="stable")
        ws, wrs = np.tile(w[sig], 2), np.tile((w * r)[sig], 2)
        c0 = np.concatenate([[0.0], np.cumsum(ws)])
        c1 = np.concatenate([[0.0], np.cumsum(wrs)])
        best = np.inf
        for jd, d in enumerate((3, 8)):
            sw = c0[d:d + n] - c0[:n]                       # Eq. 14 via cumulative sums
            swr = c1[d:d + n] - c1[:n]
            dchi = np.where(swr > 0, -swr ** 2 / sw, 0.0)   # BLS: chi2 = chi0 - (sum wr)^2/sum w
            k = int(np.argmin(dchi))
            if dchi[k] < best:
                best, arg, depth = dchi[k], (jd, k), swr[k] / sw[k]
        assert abs(res.chi2[ip] - (chi0 + best)) < 1e-11 * chi0
        assert (res.best["dur_idx"][ip], res.best["start"][ip]) == arg
        assert abs(res.best["depth"][ip] / depth - 1) < 1e-12
        if not hetero:                                       # uniform dy: deepest window wins
            d = (3, 8)[arg[0]]
            means = (c1[d:d + n] - c1[:n]) / (c0[d:d + n] - c0[:n])
            assert arg[1] == int(np.argmax(means))


# ------------------------------------------------------------------------------ P3
def test_injected_transit_recovered_on_c1():
    w = gi.make_workload(1)
    res = oracle.search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, w.tmpl, dt0=0.05)
    s = oracle.sde(res.chi2, 151)
    ib = s.best_period_idx
    truth = w.lc.meta
    step = abs(w.periods[ib] - w.periods[ib + 1])
    assert abs(w.periods[ib] - truth["period"]) <= 1.5 * step
    assert s.sde_argmax == ib and s.sde_raw[ib] > 9.0
    dt = (res.best["t0"][ib] - truth["t0"]) % truth["period"]
    dt = min(dt, truth["period"] - dt)
    assert dt < truth["t14"]
    assert 0.5 * truth["depth"] < res.best["depth"][ib] < 1.5 * truth["depth"]


# ------------------------------------------------------------------------------ P7
def test_invariants_shuffle_scale_shift(tmpl512):
    rng = np.random.default_rng(21)
    n = 80
    t = np.sort(rng.uniform(0, 30, n))
    y = 1.0 + rng.normal(0, 1e-3, n)
    dy = 1e-3 * rng.uniform(0.5, 2, n)
    periods = np.array([1.3, 4.4, 13.0])
    qs = np.array([0.05, 0.11, 0.2])
    base = oracle.search(t, y, dy, periods, qs, tmpl512, dt0=0.0)
    # (i) input order shuffle
    p = rng.permutation(n)
    sh = oracle.search(t[p], y[p], dy[p], periods, qs, tmpl512, dt0=0.0)
    assert np.allclose(sh.chi2, base.chi2, rtol=1e-13, atol=0)
    assert np.array_equal(sh.best["dur_idx"], base.best["dur_idx"])
    assert np.array_equal(sh.best["start"], base.best["start"])
    assert np.array_equal(sh.best["t0"], base.best["t0"])
    # (iii) dy -> 2^k dy scales chi2 by 4^-k exactly
    sc = oracle.search(t, y, dy * 8.0, periods, qs, tmpl512, dt0=0.0)
    assert np.array_equal(sc.chi2 * 64.0, base.chi2)
    assert np.array_equal(sc.best["start"], base.best["start"])
    assert np.array_equal(sc.best["depth"], base.best["depth"])
    # (ii) t -> t + c rotates the folded curve; stride 1 sees the same set of windows
    sf = oracle.search(t + 0.377, y, dy, periods, qs, tmpl512, dt0=0.0)
    assert np.allclose(sf.chi2, base.chi2, rtol=1e-12, atol=0)
    assert np.array_equal(sf.best["dur_idx"], base.best["dur_idx"])
    assert np.allclose(sf.best["t0"], base.best["t0"] + 0.377, rtol=0, atol=1e-12)


def test_flat_curve_is_degenerate(tmpl512):
    t = np.linspace(0, 10, 40)
    res = oracle.search(t, np.ones(40), np.full(40, 1e-3), [1.1, 2.2], [0.1, 0.2], tmpl512, dt0=0.0)
    assert np.all(res.chi2 == 0.0)
    assert np.all(res.best["dur_idx"] == 0) and np.all(res.best["start"] == 0)   # reading G22
    assert oracle.sde(res.chi2, 3).degenerate


def test_brightening_only_scores_chi2_null(tmpl512):
    rng = np.random.default_rng(5)
    t = np.sort(rng.uniform(0, 10, 40))
    y = 1.0 + np.abs(rng.normal(0, 1e-3, 40))            # every window mean is above 1
    res = oracle.search(t, y, np.full(40, 1e-3), [1.7], [0.1, 0.3], tmpl512, dt0=0.0)
    assert res.chi2[0] == res.chi2_null and res.best["depth"][0] == 0.0   # reading G7
    assert (res.best["dur_idx"][0], res.best["start"][0]) == (0, 0)


# ------------------------------------------------------------------------------ P11
def test_stride_subset_never_beats_exhaustive(tmpl512):
    w = gi.make_workload(1).subset(200)
    full = oracle.search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, w.tmpl, dt0=0.0)
    for dt0 in (0.01, 0.05, 0.1):
        sub = oracle.search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, w.tmpl, dt0=dt0)
        assert np.all(sub.chi2 >= full.chi2)
        assert sub.windows <= full.windows
    again = oracle.search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, w.tmpl, dt0=1e-9)
    assert np.array_equal(again.chi2, full.chi2)          # floor(D*dt0)=0 -> stride 1


# ------------------------------------------------------------------------------ P13
@pytest.mark.parametrize("d,s", [(9, 5), (17, 70), (30, 0)])
def test_noise_free_folded_construction(d, s, tmpl512):
    rng = np.random.default_rng(31)
    n = 75
    t = np.sort(rng.uniform(0, 40, n))
    period, a = 3.1, 2.5e-3
    _, perm = oracle.fold_sort(t, [period], want_phase=False)
    sig = perm[0]
    g, gbar = oracle.resample_template(tmpl512, d)
    y = np.ones(n)
    for j in range(d):
        y[sig[(s + j) % n]] = 1.0 - a * g[j]              # wraps for s=70
    dy = np.full(n, 1e-3)
    qs = np.array([4.5, 9.5, 17.5, 30.5]) / n
    res = oracle.search(t, y, dy, [period, 2.0], qs, tmpl512, dt0=0.0)
    assert res.chi2[0] < 1e-20 * res.chi2_null or res.chi2[0] < 1e-18
    assert res.best["dur_idx"][0] == {9: 1, 17: 2, 30: 3}[d] and res.best["start"][0] == s
    assert abs(res.best["depth"][0] / a - 1.0) < 1e-12
    assert res.best["t0"][0] == t[sig[(s + (d - 1) // 2) % n]]
    assert res.chi2[1] > 1e-3 * res.chi2_null              # wrong period does not fit


# ------------------------------------------------------------------------------ P14
def test_top_k(tmpl512):
    t, y, dy = _tiny_curve(41, n=70, hetero=False)
    periods = np.array([1.9, 6.1])
    qs = np.array([0.06, 0.13])
    full = oracle.search(t, y, dy, periods, qs, tmpl512, dt0=0.0)
    allk = oracle.search(t, y, dy, periods, qs, tmpl512, dt0=0.0, top_k=70)
    assert np.array_equal(allk.chi2, full.chi2) and np.array_equal(allk.best, full.best)
    k1 = oracle.search(t, y, dy, periods, qs, tmpl512, dt0=0.0, top_k=1)
    assert np.all(k1.chi2 >= full.chi2) and k1.windows == 2 * 2
    box = np.ones(8)                                       # box + uniform dy: deepest == best
    fb = oracle.search(t, y, dy, periods, qs, box, dt0=0.0)
    kb = oracle.search(t, y, dy, periods, qs, box, dt0=0.0, top_k=1)
    assert np.array_equal(fb.chi2, kb.chi2) and np.array_equal(fb.best, kb.best)


# ------------------------------------------------------------------------------ out_gap (runner-up)
@pytest.mark.parametrize("seed,dt0", [(3, 0.0), (4, 0.0), (5, 0.3)])
def test_gap_is_second_smallest_distinct_score_minus_best(seed, dt0, tmpl512):
    """`gap` (Best::second - best, used by the GPU parity tests' near-tie rule) against a brute force
    over ALL (duration, start) scores built from the literal per-window export: the smallest score
    strictly above the minimum, minus the minimum.  A duplicate duration (same D, bit-identical
    scores) must not count as a runner-up."""
    t, y, dy = _tiny_curve(seed, n=56)
    n = t.size
    periods = np.array([1.3, 2.9, 7.7])
    qs = np.array([3.2 / n, 6.5 / n, 6.6 / n, 11.0 / n, 20.0 / n])     # D = 3, 6, 6 (duplicate), 11, 20
    res = oracle.search(t, y, dy, periods, qs, tmpl512, dt0=dt0)
    chi0 = oracle.chi2_null(y, dy)
    for ip, period in enumerate(periods):
        scores = []
        for q in qs:
            _, _, c_out, c_in = oracle.window_chi2_literal(t, y, dy, period, q, tmpl512, dt0)
            scores.append(c_out + c_in)
        s = np.sort(np.concatenate(scores))
        best = s[0]
        # the literal export and the search differ by rounding (~1e-13 chi2): "distinct" = further
        # apart than that; the duplicate-D pair and any exact repeats of the minimum fall inside it
        above = s[s > best + 1e-11 * chi0]
        assert above.size > 0
        expect = above[0] - best
        assert abs(res.chi2[ip] - best) <= 1e-12 * chi0
        assert abs(res.gap[ip] - expect) <= 2e-11 * chi0 + 1e-9 * expect, (ip, res.gap[ip], expect)
        assert res.gap[ip] > 0.0


def test_gap_is_infinite_when_every_score_is_equal(tmpl512):
    """Flat curve: every window scores exactly chi2_0 = 0, so there is no runner-up (reading G22)."""
    t = np.linspace(0.0, 10.0, 40)
    res = oracle.search(t, np.ones(40), np.full(40, 1e-3), [1.1, 2.3], [0.1, 0.2], tmpl512, dt0=0.0)
    assert np.all(np.isinf(res.gap)) and np.all(res.chi2 == 0.0)


def test_gap_of_a_constructed_two_window_problem(tmpl512):
    """Two dips of different depth, one duration, stride = D: the runner-up is the shallower dip's
    window and the gap equals the difference of their closed-form box scores (constant template:
    score = -(sum w r)^2 / sum w)."""
    n = 40
    t = np.arange(n, dtype=np.float64)                   # period 40 -> phases i/40, identity order
    y = np.ones(n)
    y[8:12] = 1.0 - 3e-3
    y[24:28] = 1.0 - 2e-3
    dy = np.full(n, 1e-3)
    box = np.ones(16)
    res = oracle.search(t, y, dy, [40.0], [4.0 / n], box, dt0=1.0)      # D = 4, stride 4: starts 0, 4, ..
    w = 1.0 / dy[0] ** 2
    s_deep = -(4 * w * 3e-3) ** 2 / (4 * w)
    s_shallow = -(4 * w * 2e-3) ** 2 / (4 * w)
    assert res.best["start"][0] == 8 and res.best["dur_idx"][0] == 0
    assert abs(res.gap[0] - (s_shallow - s_deep)) <= 1e-12 * abs(s_deep)
