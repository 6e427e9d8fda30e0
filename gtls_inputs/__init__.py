"""Seeded synthetic inputs for the TLS/GTLS period-search hot path.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
product (``paper_2607_00348_b200/``).  It produces *inputs* only -- light curves,
the transit template array and the period / duration grids that the C-ABI call
takes as arguments -- and holds none of the search arithmetic (no folding,
sorting, window sums, chi^2, SR or SDE).

Recipes follow SURVEY.md section 8(d) / DESIGN.md "Input recipe"; the shapes stand
in for the paper's batman / Kepler inputs, which are not
available offline.
"""
from .lightcurves import (  # noqa: F401
    CADENCE_DAYS,
    BASE_SEED,
    LightCurve,
    Workload,
    make_lightcurve,
    make_workload,
    survey_curve_params,
    quad_ld_deficit,
    transit_template,
    heteroscedastic_dy,
)
from .grids import (  # noqa: F401
    G_SI,
    M_SUN,
    R_SUN,
    SECONDS_PER_DAY,
    K_MIN_GTLS,
    K_MAX_GTLS,
    Q_CAP_GTLS,
    roche_fmax_hz,
    ofir_period_grid,
    duration_grid,
    duration_k_from_eq7,
)
