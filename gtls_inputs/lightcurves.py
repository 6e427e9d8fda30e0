"""Seeded synthetic Kepler-like light curves, the transit template, and the five workloads.

Recipe: SURVEY.md section 8(d) (restated in DESIGN.md "Input recipe").  Every array is made
on the host with ``numpy.random.default_rng(seed)``, ``seed = BASE_SEED + 1000*cfg + curve``,
and is fed unchanged to both the oracle and the CUDA library.

The transit shape is a quadratic limb-darkened occultation computed by direct numerical
integration of the occulted intensity (batman is not available offline); it is input data,
not part of the search.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np
from scipy.signal import lfilter

from . import grids

CADENCE_DAYS = 29.4 / 1440.0
BASE_SEED = 260700348
LD_U1 = 0.4804
LD_U2 = 0.1867


# --------------------------------------------------------------------------------------
# transit shape (input data)
# --------------------------------------------------------------------------------------
_GL_X, _GL_W = np.polynomial.legendre.leggauss(96)


def quad_ld_deficit(z, p: float, u1: float = LD_U1, u2: float = LD_U2) -> np.ndarray:
    """Fractional flux deficit of a star with quadratic limb darkening occulted by a dark
    disk of radius ``p`` (stellar radii) centred at projected separation ``z``.

    I(mu) = 1 - u1 (1-mu) - u2 (1-mu)^2, mu = sqrt(1-r^2).  The occulted flux is
    int I(r) * arc(r) dr over the annuli r in [max(0,z-p), min(1,z+p)], where arc(r) is the
    length of the circle of radius r lying inside the occulting disk.  Gauss-Legendre in
    phi with r = lo + (hi-lo)(1-cos phi)/2 removes the square-root end-point behaviour.
    """
    z = np.abs(np.atleast_1d(np.asarray(z, dtype=np.float64)))
    out = np.zeros_like(z)
    active = z < 1.0 + p
    if not np.any(active):
        return out
    za = z[active]
    lo = np.maximum(0.0, za - p)
    hi = np.minimum(1.0, za + p)
    # split at the kink r = p - z (inside it the annuli are fully covered) when z < p
    mid = np.clip(p - za, lo, hi)
    phi = 0.5 * math.pi * (_GL_X + 1.0)                      # [K] in (0, pi)
    wphi = 0.5 * math.pi * _GL_W
    zz = za[:, None]
    occ = np.zeros_like(za)
    for a, b in ((lo, mid), (mid, hi)):
        r = a[:, None] + (b - a)[:, None] * 0.5 * (1.0 - np.cos(phi))[None, :]
        drdphi = (b - a)[:, None] * 0.5 * np.sin(phi)[None, :]
        mu = np.sqrt(np.clip(1.0 - r * r, 0.0, None))
        inten = 1.0 - u1 * (1.0 - mu) - u2 * (1.0 - mu) ** 2
        with np.errstate(divide="ignore", invalid="ignore"):
            cosang = (r * r + zz * zz - p * p) / (2.0 * r * zz)
        cosang = np.where(np.isfinite(cosang), cosang, -1.0)
        ang = 2.0 * np.arccos(np.clip(cosang, -1.0, 1.0))    # angular extent inside the disk
        ang = np.where(r + zz <= p, 2.0 * math.pi, ang)      # annulus fully covered
        occ += np.sum(inten * ang * r * drdphi * wphi[None, :], axis=1)
    total = math.pi * (1.0 - u1 / 3.0 - u2 / 6.0)
    out[active] = occ / total
    return out


def transit_template(n_tmpl: int = 512, rp_rs: float = 0.1, u1: float = LD_U1,
                     u2: float = LD_U2) -> np.ndarray:
    """Template deficit on ``n_tmpl`` nodes u_k = k/(n_tmpl-1) spanning first to fourth
    contact of a central (b=0) transit; end nodes 0, peak normalised to 1 (reading G13)."""
    u = np.linspace(0.0, 1.0, n_tmpl)
    z = (1.0 + rp_rs) * np.abs(2.0 * u - 1.0)
    g = quad_ld_deficit(z, rp_rs, u1, u2)
    g[0] = 0.0
    g[-1] = 0.0
    return np.ascontiguousarray(g / g.max())


# --------------------------------------------------------------------------------------
# light curves
# --------------------------------------------------------------------------------------
@dataclass
class LightCurve:
    t: np.ndarray
    y: np.ndarray
    dy: np.ndarray
    meta: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.t.shape[0])


def _gap_mask(n: int, starts, lengths) -> np.ndarray:
    keep = np.ones(n, dtype=bool)
    for s, l in zip(starts, lengths):
        s = int(max(0, min(n, s)))
        keep[s:min(n, s + int(l))] = False
    return keep


def _ar1(rng: np.random.Generator, n: int, phi: float, sigma_stationary: float) -> np.ndarray:
    if sigma_stationary <= 0.0:
        return np.zeros(n)
    eps = rng.normal(0.0, sigma_stationary * math.sqrt(1.0 - phi * phi), n)
    x0 = rng.normal(0.0, sigma_stationary)
    zi = np.array([phi * x0])
    x, _ = lfilter([1.0], [1.0, -phi], eps, zi=zi)
    return x


def _kepler_t14_days(period_days: float) -> float:
    return (13.0 / 24.0) * (period_days / 365.25) ** (1.0 / 3.0)


def _inject(t: np.ndarray, period: float, t0: float, t14: float, rp_rs: float,
            peak_depth: float | None) -> np.ndarray:
    """Deficit (>=0) of a strictly periodic central transit sampled at times ``t``."""
    ph = (t - t0 + 0.5 * period) % period - 0.5 * period      # time from nearest mid-transit
    z = (1.0 + rp_rs) * np.abs(ph) / (0.5 * t14)
    d = quad_ld_deficit(z, rp_rs)
    if peak_depth is not None:
        d = d * (peak_depth / float(quad_ld_deficit(np.array([0.0]), rp_rs)[0]))
    return d


def make_lightcurve(span_days: float, seed: int, sigma_white: float, sigma_red: float = 0.0,
                    phi: float = 0.9, gap_recipe: str = "none", period: float | None = None,
                    t14: float | None = None, rp_rs: float = 0.05, peak_depth: float | None = None,
                    ) -> LightCurve:
    rng = np.random.default_rng(seed)
    n_full = int(round(span_days / CADENCE_DAYS))
    t_full = np.arange(n_full, dtype=np.float64) * CADENCE_DAYS
    # gaps -------------------------------------------------------------------------------
    if gap_recipe == "none":
        keep = np.ones(n_full, dtype=bool)
    elif gap_recipe == "two_blocks":          # two contiguous blocks of 2.5 % each
        blk = int(round(0.025 * n_full))
        s1 = int(rng.integers(0, n_full // 2 - blk))
        s2 = int(rng.integers(n_full // 2, n_full - blk))
        keep = _gap_mask(n_full, [s1, s2], [blk, blk])
    elif gap_recipe == "quarters":            # one block at each of 16 quarter boundaries, 9.7 %
        frac = rng.dirichlet(np.full(16, 8.0)) * 0.097
        lengths = np.maximum(1, np.round(frac * n_full)).astype(int)
        centres = (np.arange(1, 17) * n_full) // 17
        keep = _gap_mask(n_full, centres - lengths // 2, lengths)
    elif gap_recipe == "thirty_blocks":       # 30 seeded contiguous blocks summing to 10 %
        frac = rng.dirichlet(np.full(30, 4.0)) * 0.10
        lengths = np.maximum(1, np.round(frac * n_full)).astype(int)
        slots = (np.arange(30) * n_full) // 30
        starts = slots + (rng.random(30) * (n_full // 30 - lengths).clip(min=1)).astype(int)
        keep = _gap_mask(n_full, starts, lengths)
    else:
        raise ValueError(gap_recipe)
    # noise on the ungapped cadence grid ---------------------------------------------------
    white = rng.normal(0.0, sigma_white, n_full)
    red = _ar1(rng, n_full, phi, sigma_red)
    # transit --------------------------------------------------------------------------------
    meta = {"seed": seed, "span_days": span_days, "sigma_white": sigma_white, "sigma_red": sigma_red}
    deficit = np.zeros(n_full)
    if period is not None:
        t0 = float(rng.random() * period)
        t14 = _kepler_t14_days(period) if t14 is None else t14
        deficit = _inject(t_full, period, t0, t14, rp_rs, peak_depth)
        meta.update({"period": period, "t0": t0, "t14": t14, "rp_rs": rp_rs,
                     "depth": float(deficit.max())})
    flux = 1.0 - deficit + white + red
    t = np.ascontiguousarray(t_full[keep])
    y = flux[keep]
    y = np.ascontiguousarray(y / y.mean())
    dy = np.full_like(y, sigma_white)
    return LightCurve(t, y, dy, meta)


def heteroscedastic_dy(lc: LightCurve, seed: int) -> LightCurve:
    """Parity-test variant: dy_i = sigma_w * U(0.5, 2)."""
    rng = np.random.default_rng(seed)
    dy = lc.dy * rng.uniform(0.5, 2.0, lc.n)
    return LightCurve(lc.t.copy(), lc.y.copy(), np.ascontiguousarray(dy), dict(lc.meta, hetero=True))


# --------------------------------------------------------------------------------------
# workloads c1..c5
# --------------------------------------------------------------------------------------
@dataclass
class Workload:
    name: str
    lc: LightCurve
    periods: np.ndarray          # [n_per] days, ascending frequency
    durations: np.ndarray        # [n_per, n_dur] fractions T14/P
    tmpl: np.ndarray             # [n_tmpl] deficit template
    dt0: float = 0.05

    @property
    def n_per(self) -> int:
        return int(self.periods.shape[0])

    @property
    def n_dur(self) -> int:
        return int(self.durations.shape[1])

    @property
    def trials(self) -> int:
        return self.n_per * self.n_dur

    def subset(self, every: int, offset: int = 0) -> "Workload":
        """Deterministic period subset (every k-th period) for bounded oracle runs."""
        sel = slice(offset, None, every)
        return Workload(f"{self.name}[{offset}::{every}]", self.lc,
                        np.ascontiguousarray(self.periods[sel]),
                        np.ascontiguousarray(self.durations[sel]), self.tmpl, self.dt0)


_RE_RS = grids.R_EARTH / grids.R_SUN

_CFG = {
    1: dict(span=30.0, n_dur=20, sw=1000e-6, sr=0.0, gaps="none", period=3.7, t14=2.5 / 24.0,
            rp_rs=math.sqrt(2000e-6), peak_depth=2000e-6),
    2: dict(span=90.0, n_dur=25, sw=300e-6, sr=100e-6, gaps="two_blocks", period=11.2,
            rp_rs=1.5 * _RE_RS),
    3: dict(span=1470.0, n_dur=30, sw=150e-6, sr=50e-6, gaps="quarters", period=127.0,
            rp_rs=1.0 * _RE_RS),
    4: dict(span=3000.0, n_dur=30, sw=200e-6, sr=70e-6, gaps="thirty_blocks", period=213.0,
            rp_rs=2.0 * _RE_RS),
}


def survey_curve_params(curve: int) -> dict:
    """c5: per-curve parameters drawn from the curve's own seed."""
    rng = np.random.default_rng(BASE_SEED + 1000 * 5 + curve + 7_000_000)
    sw = float(np.exp(rng.uniform(math.log(100e-6), math.log(2000e-6))))
    p = dict(span=90.0, n_dur=25, sw=sw, sr=sw / 3.0, gaps="two_blocks")
    period = float(rng.uniform(0.5, 40.0))
    rp = float(rng.uniform(0.8, 4.0))
    if curve % 2 == 0:                       # half with injected transits, half noise only
        p.update(period=period, rp_rs=rp * _RE_RS)
    return p


def make_workload(cfg: int, curve: int = 0, n_tmpl: int = 512, dt0: float = 0.05,
                  hetero: bool = False, p_min_days: float = 0.5) -> Workload:
    """Build workload c<cfg> (BASELINE.json configs[cfg-1]); ``curve`` selects the curve of c5."""
    c = dict(_CFG[cfg]) if cfg in _CFG else survey_curve_params(curve)
    seed = BASE_SEED + 1000 * cfg + curve
    lc = make_lightcurve(c["span"], seed, c["sw"], c["sr"], gap_recipe=c["gaps"],
                         period=c.get("period"), t14=c.get("t14"), rp_rs=c.get("rp_rs", 0.05),
                         peak_depth=c.get("peak_depth"))
    if hetero:
        lc = heteroscedastic_dy(lc, seed + 500)
    periods = grids.ofir_period_grid(c["span"], p_min_days=p_min_days)
    durations = grids.duration_grid(periods, c["n_dur"])
    tmpl = transit_template(n_tmpl)
    name = f"c{cfg}" + (f".{curve}" if cfg == 5 else "") + ("h" if hetero else "")
    return Workload(name, lc, periods, durations, tmpl, dt0)
