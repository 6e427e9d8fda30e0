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
