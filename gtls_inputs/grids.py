"""Period and duration grids that are *inputs* to the search call.

Period grid: Ofir (2014) cubic frequency sampling, PAPER.md:77-120 (Eq. 1-6).
Duration grid: per-period envelope k_min P^(-2/3) <= T14/P <= min(k_max P^(-2/3), cap),
PAPER.md:132-159 (Eq. 7-9), log-spaced (reading G12).

These are host-side helpers that build the workloads; both the oracle and the
CUDA library receive their output as plain arrays.
"""
from __future__ import annotations

import math

import numpy as np

# Physical constants (SI).  CODATA G, IAU nominal solar values.
G_SI = 6.67430e-11
M_SUN = 1.98847e30
R_SUN = 6.957e8
R_JUP = 7.1492e7
R_EARTH = 6.371e6
SECONDS_PER_DAY = 86400.0

# GTLS defaults.
K_MIN_GTLS = 20.05   # s^(2/3)
K_MAX_GTLS = 620.84  # s^(2/3)
Q_CAP_GTLS = 0.15
# TLS (H19) values quoted by the paper.
K_MIN_TLS = 41.39
K_MAX_TLS = 546.94
Q_CAP_TLS = 0.112


def roche_fmax_hz(r_star: float = 1.0, m_star: float = 1.0) -> float:
    """Eq. 3: f_max = 1/(2 pi) sqrt(G M / (3R)^3), in Hz."""
    gm = G_SI * m_star * M_SUN
    a_min = 3.0 * r_star * R_SUN
    return math.sqrt(gm / a_min**3) / (2.0 * math.pi)


def ofir_constants(span_days: float, r_star: float = 1.0, m_star: float = 1.0,
                   oversampling: float = 3.0, p_min_days: float | None = None):
    """A, C, N of Eq. 4-6, reading G21: S = time span in seconds."""
    span_s = span_days * SECONDS_PER_DAY
    gm = G_SI * m_star * M_SUN
    a_coef = ((2.0 * math.pi) ** (2.0 / 3.0) / math.pi) * (r_star * R_SUN) / gm ** (1.0 / 3.0) \
        / (span_s * oversampling)                                       # Eq. 5
    f_min = 2.0 / span_s                                                # Eq. 1
    f_max = roche_fmax_hz(r_star, m_star) if p_min_days is None \
        else 1.0 / (p_min_days * SECONDS_PER_DAY)
    c_coef = f_min ** (1.0 / 3.0) - a_coef / 3.0
    n_exact = (f_max ** (1.0 / 3.0) - f_min ** (1.0 / 3.0) + a_coef / 3.0) * 3.0 / a_coef  # Eq. 6
    return a_coef, c_coef, n_exact, f_min, f_max


def ofir_period_grid(span_days: float, r_star: float = 1.0, m_star: float = 1.0,
                     oversampling: float = 3.0, p_min_days: float | None = None) -> np.ndarray:
    """Trial periods in days, in ascending-frequency order (longest period first).

    f_i = (A/3 i + C)^3, i = 1..N (Eq. 4); N = ceil(Eq. 6).  The first period is
    span/2 (Eq. 1) and the last is ~P_min.
    """
    a_coef, c_coef, n_exact, _, _ = ofir_constants(span_days, r_star, m_star, oversampling, p_min_days)
    n = int(math.ceil(n_exact))
    i = np.arange(1, n + 1, dtype=np.float64)
    f = (a_coef / 3.0 * i + c_coef) ** 3
    return 1.0 / f / SECONDS_PER_DAY


def duration_k_from_eq7(r_star: float, m_star: float, r_planet_m: float = 0.0) -> float:
    """Eq. 7 rewritten as T14/P <= k P^(-2/3); returns k in s^(2/3)."""
    gm = G_SI * m_star * M_SUN
    return (r_star * R_SUN + r_planet_m) * (4.0 / (math.pi * gm)) ** (1.0 / 3.0)


def duration_grid(periods_days: np.ndarray, n_dur: int, k_min: float = K_MIN_GTLS,
                  k_max: float = K_MAX_GTLS, q_cap: float = Q_CAP_GTLS) -> np.ndarray:
    """[n_per, n_dur] duration fractions q = T14/P, log-spaced per period (reading G12).

    Lower edge k_min P^(-2/3) (Eq. 9), upper edge min(k_max P^(-2/3), q_cap) (Eq. 8 and
    PAPER.md:159), P in seconds.
    """
    p_s = np.asarray(periods_days, dtype=np.float64) * SECONDS_PER_DAY
    scale = p_s ** (-2.0 / 3.0)
    q_lo = np.minimum(k_min * scale, q_cap)
    q_hi = np.minimum(k_max * scale, q_cap)
    x = np.linspace(0.0, 1.0, n_dur, dtype=np.float64)[None, :]
    q = np.exp(np.log(q_lo)[:, None] * (1.0 - x) + np.log(q_hi)[:, None] * x)
    return np.ascontiguousarray(q)
