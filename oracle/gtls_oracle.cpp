// =====================================================================================
// TEST INFRASTRUCTURE -- NOT THE PRODUCT.
//
// Plain, slow, fp64 CPU oracle for the TLS / GTLS period search of arxiv/paper_2607_00348,
// written step by step from PAPER.md (the paper text) with the readings listed in
// DESIGN.md ("Readings of the paper", G1..G22).  It shares no code, header, table or
// helper with the CUDA path in paper_2607_00348_b200/ and neither imports the other.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may load this library.
//
// No blocking, fusion, prefix sums or padding tricks: circular indexing and direct sums,
// so that each function can be checked against the paper by eye.  OpenMP is used only
// as an outer `parallel for` over independent trial periods.
//
// Build: g++ -O2 -std=c++17 -fopenmp -ffp-contract=off -fPIC -shared (oracle/build.py).
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): P1 brute force vs the literal padded
// Eq. 15 + Eq. 16 - Eq. 11 form; P2 closed-form box case; P3 injected-transit recovery;
// P4 fold; P5 sort vs numpy stable argsort + constructed ties; P6 window sums vs cumsum;
// P7 invariants; P8 template resampling; P9/P10 SDE vs closed forms / scipy median filter;
// P11 stride example of PAPER.md:291; P13 noise-free folded-domain construction;
// P14 top-K; P12 grids (paper-printed f_max, N ~ 190 000, k values; S/2 first period).
// Parity unpinned: behaviour for n < 3 and D = n-1 (fixed only by this text).
// =====================================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <numeric>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// Eq. 10: p_i = t_i/P - floor(t_i/P), one IEEE division (reading G1).
inline double fold_phase(double t, double period) {
    const double q = t / period;
    return q - std::floor(q);
}

// PAPER.md:185 "sorted according to these phases"; ties keep ascending original index
// (reading G2) == stable sort.
void phase_order(const double* t, int64_t n, double period, std::vector<double>& phase,
                 std::vector<int32_t>& sigma) {
    phase.resize(n);
    sigma.resize(n);
    for (int64_t i = 0; i < n; ++i) phase[i] = fold_phase(t[i], period);
    std::iota(sigma.begin(), sigma.end(), 0);
    std::stable_sort(sigma.begin(), sigma.end(),
                     [&](int32_t a, int32_t b) { return phase[a] < phase[b]; });
}

// D = number of folded points inside one transit duration (reading G11):
// D = floor(q*N) clamped to [1, N-1].
inline int64_t points_in_duration(double q, int64_t n) {
    int64_t d = (int64_t)std::floor(q * (double)n);
    if (d < 1) d = 1;
    if (d > n - 1) d = n - 1;
    return d;
}

// Eq. 18: N_skip = n_IT * dt0, reading G9: stride = max(1, floor(D*dt0)).
inline int64_t t0_stride(int64_t d, double dt0) {
    if (!(dt0 > 0.0)) return 1;
    int64_t s = (int64_t)std::floor((double)d * dt0);
    return s < 1 ? 1 : s;
}

// PAPER.md:51 "calculating the number of data points in the transit signal and the flux of
// each point" (readings G13, G14): template deficit resampled to D points by linear
// interpolation at cell centres u = (j+1/2)/D over nodes k/(n_tmpl-1).  Returns mean(g).
double resample_template(const double* tmpl, int32_t n_tmpl, int64_t d, double* g) {
    double sum = 0.0;
    for (int64_t j = 0; j < d; ++j) {
        const double u = ((double)j + 0.5) / (double)d * (double)(n_tmpl - 1);
        int64_t k = (int64_t)std::floor(u);
        if (k > n_tmpl - 2) k = n_tmpl - 2;
        if (k < 0) k = 0;
        const double frac = u - (double)k;
        g[j] = tmpl[k] + frac * (tmpl[k + 1] - tmpl[k]);
        sum += g[j];
    }
    return sum / (double)d;
}

struct Best {
    double dchi2 = 0.0;      // chi2 - chi2_0 of the best candidate
    double second = std::numeric_limits<double>::infinity();  // smallest dchi2 strictly above best
    int32_t dur_idx = 0;
    int32_t start = 0;
    double depth = 0.0;
    bool any = false;
};

// Lexicographic argmin on (dchi2, jd, s): candidates arrive in ascending (jd, s) order, so a
// strict '<' keeps the first of any exact tie.
inline void offer(Best& b, double d, int32_t jd, int32_t s, double depth) {
    if (!b.any) {
        b.any = true; b.dchi2 = d; b.dur_idx = jd; b.start = s; b.depth = depth;
        return;
    }
    if (d < b.dchi2) {
        b.second = b.dchi2;
        b.dchi2 = d; b.dur_idx = jd; b.start = s; b.depth = depth;
    } else if (d > b.dchi2 && d < b.second) {
        b.second = d;
    }
}

struct Curve {
    int64_t n;
    std::vector<double> w, r;   // w_i = 1/dy_i^2, r_i = 1 - f_i (flux deficit)
    double chi2_0;              // sum_i w_i r_i^2: chi^2 of the no-transit model
};

Curve make_curve(const double* y, const double* dy, int64_t n) {
    Curve c;
    c.n = n;
    c.w.resize(n);
    c.r.resize(n);
    double s = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        c.w[i] = 1.0 / (dy[i] * dy[i]);
        c.r[i] = 1.0 - y[i];
        s += c.w[i] * c.r[i] * c.r[i];
    }
    c.chi2_0 = s;
    return c;
}

// One (period, duration) trial: all strided starts (or the top_k deepest), windows are the
// sorted positions (s+j) mod N, j < D  (Fig. 3 padding == circular indexing, reading G3/G4).
//   rbar  = sum w r / sum w                           (Eq. 12-14, readings G5, G6)
//   a     = max(rbar, 0) / mean(g_D)                  (Eq. 13, reading G7)
//   chi2  = sum_{i not in W} w (f-1)^2 + sum_{j<D} w (f - (1 - a g_D[j]))^2    (Eq. 15-16)
//         = chi2_0 - 2 a C + a^2 G,  C = sum_j g_j w r,  G = sum_j g_j^2 w
// (the identity is pinned by tests/test_oracle_chi2.py against the literal form below).
void scan_duration(const Curve& c, const std::vector<int32_t>& sigma, int32_t jd, int64_t d,
                   int64_t stride, const double* g, double gbar, int32_t top_k, Best& best,
                   int64_t* n_windows) {
    const int64_t n = c.n;
    std::vector<int64_t> starts;
    for (int64_t s = 0; s < n; s += stride) starts.push_back(s);
    std::vector<double> rbar(starts.size());
    for (size_t q = 0; q < starts.size(); ++q) {
        double sw = 0.0, swr = 0.0;
        for (int64_t j = 0; j < d; ++j) {
            const int32_t i = sigma[(starts[q] + j) % n];
            sw += c.w[i];
            swr += c.w[i] * c.r[i];
        }
        rbar[q] = swr / sw;
    }
    std::vector<size_t> sel(starts.size());
    std::iota(sel.begin(), sel.end(), 0);
    if (top_k > 0 && (size_t)top_k < sel.size()) {
        // K deepest windows, ties -> lower start (reading G19, pruning variant)
        std::stable_sort(sel.begin(), sel.end(), [&](size_t a, size_t b) { return rbar[a] > rbar[b]; });
        sel.resize(top_k);
        std::sort(sel.begin(), sel.end());
    }
    for (size_t q : sel) {
        const double a = std::max(rbar[q], 0.0) / gbar;
        double cc = 0.0, gg = 0.0;
        for (int64_t j = 0; j < d; ++j) {
            const int32_t i = sigma[(starts[q] + j) % n];
            cc += g[j] * (c.w[i] * c.r[i]);
            gg += (g[j] * g[j]) * c.w[i];
        }
        const double dchi2 = -2.0 * a * cc + (a * a) * gg;
        offer(best, dchi2, jd, (int32_t)starts[q], a);
        if (n_windows) ++*n_windows;
    }
}

}  // namespace

extern "C" {

struct oracle_best { int32_t dur_idx; int32_t start; double depth; double t0; };
struct oracle_summary {
    int64_t best_period_idx; int32_t best_dur_idx; int32_t best_start;
    double best_period, best_t0, best_depth, chi2_min, chi2_null, sde_raw_max, sde_max;
    int64_t sde_argmax; int64_t windows_evaluated;
};

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_fold(const double* t, int64_t n, double period, double* phase) {
    for (int64_t i = 0; i < n; ++i) phase[i] = fold_phase(t[i], period);
}

void oracle_fold_sort(const double* t, int64_t n, const double* periods, int64_t n_per,
                      double* phase_out, int32_t* perm_out) {
#pragma omp parallel for schedule(dynamic)
    for (int64_t ip = 0; ip < n_per; ++ip) {
        std::vector<double> phase;
        std::vector<int32_t> sigma;
        phase_order(t, n, periods[ip], phase, sigma);
        if (phase_out) std::memcpy(phase_out + ip * n, phase.data(), n * sizeof(double));
        std::memcpy(perm_out + ip * n, sigma.data(), n * sizeof(int32_t));
    }
}

int64_t oracle_points_in_duration(double q, int64_t n) { return points_in_duration(q, n); }
int64_t oracle_stride(int64_t d, double dt0) { return t0_stride(d, dt0); }
double oracle_resample_template(const double* tmpl, int32_t n_tmpl, int64_t d, double* g) {
    return resample_template(tmpl, n_tmpl, d, g);
}

// Literal per-window chi^2 for ONE (period, duration fraction): O(N) per window, no identity
// used.  For every strided start s it writes
//   depth[s]    = a,
//   chi2_out[s] = sum over points outside the window of w (f-1)^2        (Eq. 15 on the circle)
//   chi2_in[s]  = sum_{j<D} w (f - (1 - a g_j))^2                        (Eq. 16)
// Returns the number of starts written (arrays must hold ceil(N/stride) entries).
int64_t oracle_window_chi2_literal(const double* t, const double* y, const double* dy, int64_t n,
                                   double period, double q, const double* tmpl, int32_t n_tmpl,
                                   double dt0, int32_t* start, double* depth, double* chi2_out,
                                   double* chi2_in) {
    std::vector<double> phase;
    std::vector<int32_t> sigma;
    phase_order(t, n, period, phase, sigma);
    const int64_t d = points_in_duration(q, n);
    const int64_t stride = t0_stride(d, dt0);
    std::vector<double> g(d);
    const double gbar = resample_template(tmpl, n_tmpl, d, g.data());
    int64_t k = 0;
    std::vector<char> inwin(n);
    for (int64_t s = 0; s < n; s += stride, ++k) {
        std::fill(inwin.begin(), inwin.end(), 0);
        double sw = 0.0, swf = 0.0;
        for (int64_t j = 0; j < d; ++j) {
            const int32_t i = sigma[(s + j) % n];
            inwin[i] = 1;
            const double w = 1.0 / (dy[i] * dy[i]);
            sw += w;
            swf += w * y[i];
        }
        const double fbar = swf / sw;                  // weighted mean flux in the window
        const double a = std::max(1.0 - fbar, 0.0) / gbar;
        double out = 0.0;
        for (int64_t i = 0; i < n; ++i)
            if (!inwin[i]) { const double e = (y[i] - 1.0) / dy[i]; out += e * e; }
        double in = 0.0;
        for (int64_t j = 0; j < d; ++j) {
            const int32_t i = sigma[(s + j) % n];
            const double model = 1.0 - a * g[j];
            const double e = (y[i] - model) / dy[i];
            in += e * e;
        }
        start[k] = (int32_t)s; depth[k] = a; chi2_out[k] = out; chi2_in[k] = in;
    }
    return k;
}

// The search.  durations: [n_dur] shared, or [n_per][n_dur] when
// dur_per_period != 0.  Outputs: chi2[n_per]; best[n_per] (nullable); gap[n_per] (nullable):
// second-smallest distinct dchi2 minus the smallest (for the near-tie parity rule).
int oracle_search(const double* t, const double* y, const double* dy, int64_t n,
                  const double* periods, int64_t n_per, const double* durations, int32_t n_dur,
                  int32_t dur_per_period, const double* tmpl, int32_t n_tmpl, double dt0,
                  int32_t top_k, int32_t n_threads, double* out_chi2, oracle_best* out_best,
                  double* out_gap, int64_t* out_windows) {
    if (n < 2 || n_per < 1 || n_dur < 1 || n_tmpl < 2) return -1;
    const Curve c = make_curve(y, dy, n);
    int64_t windows_total = 0;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic) reduction(+ : windows_total)
    for (int64_t ip = 0; ip < n_per; ++ip) {
        std::vector<double> phase, g;
        std::vector<int32_t> sigma;
        phase_order(t, n, periods[ip], phase, sigma);               // steps 1-2
        Best best;
        int64_t nw = 0;
        const double* qrow = dur_per_period ? durations + ip * (int64_t)n_dur : durations;
        for (int32_t jd = 0; jd < n_dur; ++jd) {                    // step 3
            const int64_t d = points_in_duration(qrow[jd], n);
            const int64_t stride = t0_stride(d, dt0);
            g.resize(d);
            const double gbar = resample_template(tmpl, n_tmpl, d, g.data());
            scan_duration(c, sigma, jd, d, stride, g.data(), gbar, top_k, best, &nw);  // step 4
        }
        out_chi2[ip] = c.chi2_0 + best.dchi2;                       // step 5
        if (out_best) {
            const int64_t d = points_in_duration(qrow[best.dur_idx], n);
            out_best[ip].dur_idx = best.dur_idx;
            out_best[ip].start = best.start;
            out_best[ip].depth = best.depth;
            out_best[ip].t0 = t[sigma[(best.start + (d - 1) / 2) % n]];
        }
        if (out_gap) out_gap[ip] = best.second - best.dchi2;
        windows_total += nw;
    }
    if (out_windows) *out_windows = windows_total;
    return 0;
}

double oracle_chi2_null(const double* y, const double* dy, int64_t n) {
    return make_curve(y, dy, n).chi2_0;
}

// Step 6: SR, SDE_raw (Eq. 17; readings G15, G16) and the moving-median
// detrended SDE (readings G17, G18).  Returns 1 when degenerate (chi2_min == 0
// or sigma_SR == 0: SDE outputs are zero), 0 otherwise.
int oracle_sde(const double* chi2, int64_t n_per, int32_t kernel, double* sr, double* sde_raw,
               double* sde, int64_t* best_period_idx, int64_t* sde_argmax) {
    int64_t imin = 0;
    for (int64_t i = 1; i < n_per; ++i) if (chi2[i] < chi2[imin]) imin = i;
    *best_period_idx = imin;
    *sde_argmax = imin;
    const double cmin = chi2[imin];
    bool degenerate = !(cmin > 0.0);
    double mean = 0.0, var = 0.0;
    if (!degenerate) {
        for (int64_t i = 0; i < n_per; ++i) { sr[i] = cmin / chi2[i]; mean += sr[i]; }
        mean /= (double)n_per;
        for (int64_t i = 0; i < n_per; ++i) var += (sr[i] - mean) * (sr[i] - mean);
        var /= (double)n_per;                                   // population variance (G16)
        if (!(var > 0.0)) degenerate = true;
    }
    if (degenerate) {
        for (int64_t i = 0; i < n_per; ++i) { sr[i] = 0.0; sde_raw[i] = 0.0; sde[i] = 0.0; }
        return 1;
    }
    const double sd = std::sqrt(var);
    for (int64_t i = 0; i < n_per; ++i) sde_raw[i] = (sr[i] - mean) / sd;
    if (kernel <= 1) {
        for (int64_t i = 0; i < n_per; ++i) sde[i] = sde_raw[i];
    } else {
        const int64_t h = (kernel - 1) / 2;
        std::vector<double> win(kernel);
        for (int64_t i = 0; i < n_per; ++i) {
            for (int64_t k = -h; k <= h; ++k) {
                int64_t j = i + k;
                if (j < 0) j = 0;
                if (j > n_per - 1) j = n_per - 1;               // edge replication (G17)
                win[k + h] = sde_raw[j];
            }
            std::sort(win.begin(), win.end());
            sde[i] = sde_raw[i] - win[h];
        }
    }
    int64_t imax = 0;
    for (int64_t i = 1; i < n_per; ++i) if (sde[i] > sde[imax]) imax = i;
    *sde_argmax = imax;
    return 0;
}

// ---- Period and duration grids (paper section 2.2) ---------------
// SI constants: CODATA G, IAU nominal solar mass / radius.  Span and periods are in days,
// stellar radius and mass in solar units.
static const double kG = 6.67430e-11, kMsun = 1.98847e30, kRsun = 6.957e8, kDay = 86400.0;

// Eq. 3: f_max = 1/(2 pi) sqrt(G M / (3R)^3), Hz.
double oracle_roche_fmax_hz(double r_star, double m_star) {
    const double a_min = 3.0 * r_star * kRsun;
    return std::sqrt(kG * m_star * kMsun / (a_min * a_min * a_min)) / (2.0 * M_PI);
}

// Eq. 1, 5, 6, reading G21: the S of Eq. 5 is the time span in seconds
// and OS the oversampling factor.  p_min_days <= 0 takes f_max from Eq. 3.  Writes A, C, N.
void oracle_ofir_constants(double span_days, double r_star, double m_star, double oversampling,
                           double p_min_days, double* A, double* Cc, double* n_exact) {
    const double S = span_days * kDay;
    const double f_min = 2.0 / S;                                                       // Eq. 1
    const double f_max = p_min_days > 0.0 ? 1.0 / (p_min_days * kDay) : oracle_roche_fmax_hz(r_star, m_star);
    *A = std::pow(2.0 * M_PI, 2.0 / 3.0) / M_PI * (r_star * kRsun) / std::cbrt(kG * m_star * kMsun)
         / (S * oversampling);                                                          // Eq. 5
    *Cc = std::cbrt(f_min) - *A / 3.0;
    *n_exact = (std::cbrt(f_max) - std::cbrt(f_min) + *A / 3.0) * 3.0 / *A;             // Eq. 6
}

// N = ceil(Eq. 6).
int64_t oracle_period_grid_size(double span_days, double r_star, double m_star, double oversampling,
                                double p_min_days) {
    double A, Cc, n_exact;
    oracle_ofir_constants(span_days, r_star, m_star, oversampling, p_min_days, &A, &Cc, &n_exact);
    return (int64_t)std::ceil(n_exact);
}

// Eq. 4: f_i = (A/3 i + C)^3, i = 1..N; periods in days in ascending-frequency
// order (the first is S/2 by Eq. 1, the last ~P_min).  Returns N.
int64_t oracle_period_grid(double span_days, double r_star, double m_star, double oversampling,
                           double p_min_days, double* out_periods, int64_t capacity) {
    double A, Cc, n_exact;
    oracle_ofir_constants(span_days, r_star, m_star, oversampling, p_min_days, &A, &Cc, &n_exact);
    const int64_t N = (int64_t)std::ceil(n_exact);
    for (int64_t i = 1; i <= N && i <= capacity; ++i) {
        const double c = A / 3.0 * (double)i + Cc;
        const double f = c * c * c;
        out_periods[i - 1] = 1.0 / f / kDay;
    }
    return N;
}

// Eq. 8-9 with the cap of PAPER.md:159, reading G12: per period n_dur
// fractions q = T14/P log-spaced from min(k_min P^(-2/3), cap) to min(k_max P^(-2/3), cap),
// P in seconds; out[ip*n_dur + j].  n_dur = 1 gives the lower edge.
void oracle_duration_grid(const double* periods_days, int64_t n_per, int32_t n_dur, double k_min,
                          double k_max, double q_cap, double* out) {
    for (int64_t ip = 0; ip < n_per; ++ip) {
        const double scale = std::pow(periods_days[ip] * kDay, -2.0 / 3.0);
        const double q_lo = std::min(k_min * scale, q_cap), q_hi = std::min(k_max * scale, q_cap);
        for (int32_t j = 0; j < n_dur; ++j) {
            const double x = n_dur > 1 ? (double)j / (double)(n_dur - 1) : 0.0;
            out[ip * n_dur + j] = std::exp(std::log(q_lo) * (1.0 - x) + std::log(q_hi) * x);
        }
    }
}

}  // extern "C"
