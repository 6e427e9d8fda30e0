"""P12: grid helpers against the values the paper prints (tests/golden/paper_pins.json)."""
import json
import os

import numpy as np

import gtls_inputs as gi
from gtls_inputs import grids

PINS = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_pins.json")))


def test_fmax_solar_matches_paper():
    pin = PINS["f_max_hz_solar"]
    assert abs(gi.roche_fmax_hz() / pin["value"] - 1.0) < pin["rel_tol"]
    pmin = 1.0 / gi.roche_fmax_hz() / 86400.0
    assert abs(pmin - PINS["p_min_days_solar"]["value"]) < PINS["p_min_days_solar"]["abs_tol"]


def test_period_count_1500d():
    pin = PINS["n_periods_1500d"]
    p = gi.ofir_period_grid(1500.0)
    assert abs(p.size / pin["value"] - 1.0) < pin["rel_tol"]
    assert abs(p[0] - 750.0) < 1e-9                 # Eq. 1: P_max = S/2
    assert abs(p[-1] - 1.0 / gi.roche_fmax_hz() / 86400.0) < 1e-4
    assert np.all(np.diff(p) < 0)                   # ascending frequency
    # cubic sampling (Eq. 4): f^(1/3) is uniformly spaced
    c = (1.0 / p) ** (1.0 / 3.0)
    d = np.diff(c)
    assert np.allclose(d, d[0], rtol=1e-6)


def test_tls_duration_constants_fix_units():
    assert abs(gi.duration_k_from_eq7(0.13, 0.1) / PINS["k_min_tls"]["value"] - 1) < PINS["k_min_tls"]["rel_tol"]
    k = gi.duration_k_from_eq7(3.5, 1.0, 2 * grids.R_JUP)
    assert abs(k / PINS["k_max_tls"]["value"] - 1) < PINS["k_max_tls"]["rel_tol"]
    assert gi.K_MIN_GTLS == PINS["k_min_gtls"]["value"]
    assert gi.K_MAX_GTLS == PINS["k_max_gtls"]["value"]
    assert gi.Q_CAP_GTLS == PINS["q_cap_gtls"]["value"]


def test_duration_grid_envelope():
    p = gi.ofir_period_grid(90.0, p_min_days=0.5)
    q = gi.duration_grid(p, 25)
    ps = p * 86400.0
    assert q.shape == (p.size, 25)
    assert np.allclose(q[:, 0], np.minimum(20.05 * ps ** (-2 / 3), 0.15))
    assert np.allclose(q[:, -1], np.minimum(620.84 * ps ** (-2 / 3), 0.15))
    assert np.all(np.diff(q, axis=1) >= 0) and q.max() <= 0.15 + 1e-15
    r = q[:, 1:] / q[:, :-1]
    assert np.allclose(r, r[:, :1])                  # log spacing


def test_workload_shapes_match_survey_table():
    for cfg, (n, n_per, n_dur) in {1: (1469, 3052, 20), 2: (4188, 10483, 25)}.items():
        w = gi.make_workload(cfg)
        assert (w.lc.n, w.n_per, w.n_dur) == (n, n_per, n_dur)
        assert abs(w.lc.y.mean() - 1.0) < 1e-12
        w2 = gi.make_workload(cfg)
        assert np.array_equal(w.lc.y, w2.lc.y)       # seeded: reproducible


def test_template_shape():
    g = gi.transit_template(512)
    assert g[0] == 0.0 and g[-1] == 0.0 and abs(g.max() - 1.0) < 1e-15
    assert np.allclose(g, g[::-1], atol=1e-12)
    assert np.all(np.diff(g[:256]) > 0)
    # uniform-source overlap area closed form pins the occultation integrator
    import math
    z, p = 1.0, 0.1
    k1 = math.acos((1 - p * p + z * z) / (2 * z)); k0 = math.acos((p * p + z * z - 1) / (2 * p * z))
    area = (p * p * k0 + k1 - 0.5 * math.sqrt(4 * z * z - (1 + z * z - p * p) ** 2)) / math.pi
    assert abs(gi.quad_ld_deficit([1.0], 0.1, 0.0, 0.0)[0] - area) < 1e-8
    assert abs(gi.quad_ld_deficit([0.3], 0.1, 0.0, 0.0)[0] - 0.01) < 1e-10


# ---- the oracle's own grid functions (oracle/gtls_oracle.cpp), pinned to the paper's printed values,
# ---- to closed forms / invariants, and to the independent numpy generators of gtls_inputs
def test_oracle_fmax_and_count_match_paper():
    import oracle
    pin = PINS["f_max_hz_solar"]
    assert abs(oracle.roche_fmax_hz() / pin["value"] - 1.0) < pin["rel_tol"]
    p = oracle.period_grid(1500.0)                   # S = 1500 d, OS = 3 -> N ~ 190 000
    pin = PINS["n_periods_1500d"]
    assert abs(p.size / pin["value"] - 1.0) < pin["rel_tol"]
    assert abs(p[0] - 750.0) < 1e-9                  # Eq. 1: P_max = S/2 exactly (C fixes f_1 = f_min)
    assert abs(p[-1] - PINS["p_min_days_solar"]["value"]) < PINS["p_min_days_solar"]["abs_tol"]
    assert p[-1] <= 1.0 / oracle.roche_fmax_hz() / 86400.0 * (1 + 1e-12)   # N = ceil: reaches f_max
    assert np.all(np.diff(p) < 0)
    d = np.diff((1.0 / p) ** (1.0 / 3.0))            # Eq. 4: f^(1/3) uniformly spaced
    assert np.allclose(d, d[0], rtol=1e-6)


def test_oracle_period_grid_scaling_and_oversampling():
    import oracle
    a = oracle.period_grid(90.0, p_min_days=0.5)
    assert abs(a[0] - 45.0) < 1e-10 and a[-1] <= 0.5 * (1 + 1e-12) and a[-2] > 0.5
    b = oracle.period_grid(90.0, oversampling=6.0, p_min_days=0.5)
    assert abs((b.size - 1) / (a.size - 1) - 2.0) < 2e-3            # Eq. 5: A ~ 1/OS, Eq. 6: N ~ 1/A
    # Eq. 5: A ~ R / M^(1/3); a star with R = 2, M = 8 has the same A as the Sun
    c = oracle.period_grid(90.0, r_star=2.0, m_star=8.0, p_min_days=0.5)
    assert c.size == a.size and np.allclose(c, a, rtol=1e-12)
    # independent numpy implementation (gtls_inputs.grids)
    assert a.size == gi.ofir_period_grid(90.0, p_min_days=0.5).size
    assert np.allclose(a, gi.ofir_period_grid(90.0, p_min_days=0.5), rtol=1e-13, atol=0)


def test_oracle_duration_grid():
    import oracle
    p = oracle.period_grid(90.0, p_min_days=0.5)
    q = oracle.duration_grid(p, 25)
    assert q.shape == (p.size, 25) and q.max() <= 0.15 * (1 + 1e-15)
    ps = p * 86400.0
    # Eq. 8-9 in the form T14 = k P^(1/3): lower edge in seconds, cube of it is linear in P
    t14_lo = q[:, 0] * ps
    free = q[:, 0] < 0.15 * (1 - 1e-12)
    assert np.allclose(t14_lo[free] ** 3 / ps[free], PINS["k_min_gtls"]["value"] ** 3, rtol=1e-12)
    capped = q[:, -1] >= 0.15 * (1 - 1e-12)
    assert capped.any() and (~capped).any()
    assert np.allclose((q[~capped, -1] * ps[~capped]) ** 3 / ps[~capped], PINS["k_max_gtls"]["value"] ** 3, rtol=1e-12)
    r = q[:, 1:] / q[:, :-1]
    assert np.allclose(r, r[:, :1], rtol=1e-12)                      # log spacing
    assert np.allclose(q, gi.duration_grid(p, 25), rtol=1e-13, atol=0)
    assert np.allclose(oracle.duration_grid(p[:5], 1)[:, 0], q[:5, 0], rtol=1e-15)
    # TLS constants with the TLS cap
    qt = oracle.duration_grid(p, 10, 41.39, 546.94, 0.112)
    assert qt.max() <= 0.112 * (1 + 1e-15) and np.all(qt[:, 0] >= q[:, 0])
