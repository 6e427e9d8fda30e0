/*
 * gtls.h -- C ABI of libgtls: the Transit Least Squares (TLS) period search that GTLS
 * (arxiv/paper_2607_00348) accelerates, as hand-written CUDA for NVIDIA B200 (sm_100a).
 *
 * Citations are to PAPER.md (the paper text) by line, plus the readings G1..G22 listed in
 * DESIGN.md.  Every step of the search runs in CUDA kernels; there is no CPU fallback: if no
 * CUDA device is usable the calls return GTLS_ECUDA.
 *
 * Conventions
 *   - Plain C: no exceptions cross the boundary.  Return 0 (GTLS_OK) on success, a negative
 *     GTLS_E* code on error.  GTLS_EDEGENERATE is a documented partial success (see below).
 *   - Every pointer is caller-owned.  The library never frees or retains a pointer after the
 *     call returns.  Outputs are written only on success / GTLS_EDEGENERATE.
 *   - `opts->pointers_on_device == 0`: all array arguments are HOST pointers; the library
 *     allocates device memory, copies in, runs, copies out and synchronises.
 *     `opts->pointers_on_device == 1`: all array arguments (inputs and outputs, but not
 *     `opts`, `out_summary` or `opts->stats`, which are always host structs) are DEVICE
 *     pointers on `opts->device`, e.g. `torch.Tensor.data_ptr()`; work is enqueued on
 *     `opts->stream` (a cudaStream_t; NULL = the legacy default stream).  The call
 *     synchronises the stream before returning (it reads back a few validation flags and the
 *     summary), so results are complete on return.
 *   - Units: `t` and `period_grid` share one time unit (days in all shipped workloads);
 *     `duration_grid` holds dimensionless fractions q = T14 / P.
 *   - `t` need not be sorted.  The library does not normalise or detrend: `y`
 *     must already be normalised to mean ~1.
 *   - Thread safety: concurrent calls are safe when they use distinct streams and distinct
 *     workspaces (or let the library allocate its own).
 *   - Process state: every entry point makes `opts->device` the calling thread's current CUDA device
 *     (cudaSetDevice) and leaves it current on return; a caller that works on another device sets it
 *     again.  Nothing else of the caller's CUDA state is changed.
 */
#ifndef GTLS_H_
#define GTLS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GTLS_OK            0
#define GTLS_EINVAL       (-1)  /* NULL required pointer, n < 3, n_per < 1, n_dur < 1, n_tmpl < 2,
                                   even / negative sde_kernel, dt0 < 0, unknown option value     */
#define GTLS_ENONFINITE   (-2)  /* NaN / Inf in t, y, dy, or dy <= 0                            */
#define GTLS_EGRID        (-3)  /* period <= 0 or non-finite; duration fraction not in (0, 0.5]   */
#define GTLS_ENOMEM       (-4)  /* device allocation failed / caller workspace too small         */
#define GTLS_ECUDA        (-5)  /* CUDA error; text via gtls_last_cuda_error()                   */
#define GTLS_EDEGENERATE  (-6)  /* chi2_min == 0 or sigma_SR == 0: chi2 / best outputs are valid,
                                   SDE outputs are set to 0                                      */
#define GTLS_EUNSUPPORTED (-7)  /* option combination not implemented (see field comments)      */

/* Best trial of one period.  `start` is the index, in the phase-sorted
 * folded curve, of the first in-transit point; the window is sorted positions
 * (start + j) mod n, j < D, with D = clamp(floor(q * n), 1, n-1) (reading G11).
 * `depth` is the scaled template depth a = max(rbar, 0) / mean(g_D) (Eq. 12-13).
 * `t0` is the observed time of the window's middle point, t[sigma[(start + (D-1)/2) mod n]]
 * (trial mid-transit times coincide with observed points). */
typedef struct {
    int32_t dur_idx;
    int32_t start;
    double  depth;
    double  t0;
} gtls_best;

/* Optional per-stage timing / counters, filled when opts->stats != NULL (host struct).
 * Times are CUDA-event milliseconds summed over all period tiles of the call. */
typedef struct {
    double  ms_total;        /* first kernel to last kernel of the call                           */
    double  ms_pre;          /* a0: per-curve arrays, validation, duration table                  */
    double  ms_fold;         /* a1 when it runs as a kernel of its own (LSD sort path); ~0 otherwise */
    double  ms_sort;         /* general path: the fused a1-a4 stage (fold, bucket sort, gather,
                                wrap pad, prefix sums are one chain of kernels)                   */
    double  ms_scan;         /* a3+a4 when separate (LSD sort path); ~0 otherwise                  */
    double  ms_chi2;         /* a5-a8: trial binning + the ring kernels.  Fused small-N path
                                (path == 1): the ONE kernel that runs a1-a8                       */
    double  ms_reduce;       /* a8: per-period lexicographic argmin                               */
    double  ms_epilogue;     /* a9: SR, SDE_raw, median detrend, argmax                           */
    int64_t kernel_launches; /* kernels launched by this call                                     */
    int64_t chi2_launches;   /* launches of the in-transit chi2 kernel                            */
    int64_t windows;         /* (period, duration, start) windows evaluated                       */
    int64_t window_points;   /* sum over evaluated windows of D (in-transit point visits)         */
    int64_t period_points;   /* n * n_per                                                         */
    int32_t period_tile;     /* periods in flight per tile                                        */
    int32_t path;            /* 1 = fused shared-memory path, 2 = general tiled path              */
    int32_t uniform_dy;      /* 1 when all dy are equal (G is position independent)               */
    int32_t reserved;
} gtls_stats;

typedef struct {
    uint32_t struct_size;        /* sizeof(gtls_opts), for ABI versioning                         */
    double   dt0;                /* Eq. 18: stride = max(1, floor(D*dt0)); 0 => 1   */
    int32_t  top_k;              /* 0 => chi2 at every strided start (the paper's search).
                                    K in 1..8 => pruning variant (reading G19): per (period, duration)
                                    the K starts of largest running-mean depth (ties: lower start) and
                                    chi2 only there.  K > 8, or K > 0 with chi2_fp32 => GTLS_EUNSUPPORTED */
    int32_t  dur_per_period;     /* 0: duration_grid[n_dur] shared by all periods;
                                    1: duration_grid[n_per][n_dur] (row per period, reading G12)   */
    int32_t  sde_kernel;         /* odd window of the moving-median detrend (PAPER.md:279,
                                    reading G17); 0 or 1 => SDE = SDE_raw                          */
    int32_t  chi2_fp32;          /* 0 = fp64.  1 = fp32 in-transit variant: template taps, X and the
                                    window accumulators of the chi2 kernels in fp32 (<= 24 products
                                    per sum); column sums, prefix sums, depth and scoring stay fp64.
                                    chi2 within 1e-6 relative of the fp64 result (north_star: 1e-4)  */
    int32_t  pointers_on_device; /* see Conventions                                               */
    int32_t  device;             /* CUDA device ordinal                                           */
    void*    stream;             /* cudaStream_t                                                  */
    void*    workspace;          /* optional caller-owned DEVICE scratch (256-byte aligned)        */
    size_t   workspace_bytes;    /* its size; must be >= gtls_workspace_bytes(...)                 */
    int32_t  period_tile;        /* periods processed per tile; 0 = automatic                     */
    int32_t  path;               /* 0 = automatic; 1 = force the fused small-N path (one CTA per
                                    (curve, period): fold, sort, pad, scans and chi2 in shared memory),
                                    GTLS_EUNSUPPORTED where it does not apply: dy not uniform, top_k or
                                    chi2_fp32 set, n_dur > 32, a window class stride above 31 columns
                                    (dt0 below ~0.045 with long durations, or dt0 above 31 / D_max), or
                                    a light curve too long for a CTA's shared memory (n > ~8000);
                                    2 = force the general tiled path                               */
    gtls_stats* stats;           /* optional, host                                                */
} gtls_opts;

typedef struct {
    int64_t best_period_idx;     /* argmin_P chi2(P), ties -> lowest index (= argmax SDE_raw)      */
    int32_t best_dur_idx;
    int32_t best_start;
    double  best_period, best_t0, best_depth;
    double  chi2_min;            /* min_P chi2(P)                                                 */
    double  chi2_null;           /* chi2_0 = sum_i ((1 - y_i)/dy_i)^2, the no-transit model        */
    double  sde_raw_max;         /* SDE_raw at best_period_idx                                    */
    double  sde_max;             /* max_P SDE(P)                                                  */
    int64_t sde_argmax;          /* argmax_P SDE(P), ties -> lowest index                         */
    int64_t windows_evaluated;
} gtls_summary;

/* Fill `o` with the defaults used when opts == NULL: dt0 = 0.05 (the paper's worked example,
 * PAPER.md:291), top_k 0, dur_per_period 0, sde_kernel 151, fp64, host pointers, device 0,
 * default stream, no workspace, automatic tile and path. */
void gtls_opts_default(gtls_opts* o);

/* The search: for every trial period fold (Eq. 10), sort by phase (PAPER.md:185,
 * ties by original index), wrap-pad (Fig. 3), prefix sums (Eq. 14),
 * and for every duration and strided start (Eq. 18) the mean-matched depth (Eq. 12-13) and
 *   chi2 = chi2_out (Eq. 15 minus the Eq. 11 edge term) + chi2_in (Eq. 16);
 * then chi2(P) = min over (duration, start) with lexicographic tie-break (chi2, dur_idx, start),
 * SR(P) = chi2_min / chi2(P), SDE_raw (Eq. 17; population sigma) and the
 * moving-median detrended SDE.
 *
 *   t, y, dy        [n]        light curve: times, normalised flux, 1-sigma uncertainties (> 0)
 *   period_grid     [n_per]    trial periods (> 0), any order; SDE median runs in this order
 *   duration_grid   [n_dur] or [n_per][n_dur] fractions T14/P in (0, 0.5]
 *   tmpl            [n_tmpl]   transit template as a flux DEFICIT on nodes u_k = k/(n_tmpl-1)
 *                              across first..fourth contact (reading G13); resampled to D points
 *                              by linear interpolation at cell centres (j+1/2)/D (reading G14)
 *   out_chi2        [n_per]    required
 *   out_best        [n_per]    may be NULL
 *   out_sde_raw, out_sde [n_per] may be NULL
 *   out_summary     host struct, may be NULL
 */
int gtls_search(const double* t, const double* y, const double* dy, int64_t n,
                const double* period_grid, int64_t n_per,
                const double* duration_grid, int32_t n_dur,
                const double* tmpl, int32_t n_tmpl,
                const gtls_opts* opts,
                double* out_chi2, gtls_best* out_best,
                double* out_sde_raw, double* out_sde,
                gtls_summary* out_summary);

/* Two-stage hierarchical search (section 2.5).
 *   Stage 1: gtls_search over all periods with opts->dt0 (the coarse T0 skip of Eq. 18).
 *   Stage 2: the n_refine trial periods of highest SDE after stage 1 (ties -> lower index; the paper uses
 *            ~200) are searched again with stride 1 (every trial T0, "without skipping");
 *            their chi2 / best records replace the stage-1 values, then SR, SDE_raw, SDE and the summary
 *            are recomputed over the whole grid (a9).
 * Arguments as gtls_search.  out_best is required here.  out_refined [min(n_refine, n_per)] (int64
 * indices into period_grid in selection order; host or device like the other arrays) may be NULL.
 * n_refine <= 0 is GTLS_EINVAL.  A degenerate stage-1 spectrum returns GTLS_EDEGENERATE without stage 2.
 * The SNR statistic the paper mentions for stage 2 is not defined in the paper and is not computed. */
int gtls_search_two_stage(const double* t, const double* y, const double* dy, int64_t n,
                          const double* period_grid, int64_t n_per,
                          const double* duration_grid, int32_t n_dur,
                          const double* tmpl, int32_t n_tmpl,
                          const gtls_opts* opts, int32_t n_refine,
                          double* out_chi2, gtls_best* out_best,
                          double* out_sde_raw, double* out_sde,
                          int64_t* out_refined, gtls_summary* out_summary);

/* Parity / debug export of steps a5-a8 AS THE HOT KERNEL COMPUTES THEM: runs the general tiled path of
 * gtls_search (fold, sort, pad, scans, trial binning, the register-ring chi2 kernel of this trial's variant,
 * instantiated to dump its scores) for ONE (period, duration fraction q) and returns, for every strided start
 * k*stride < n (Eq. 18), the start index, the depth a (Eq. 12-13) and dchi2 = chi2(window) - chi2_0 =
 * -2 a C + a^2 G (Eq. 15 + 16 minus the Eq. 11 edge term) exactly as the kernel's scoring step saw them --
 * including every non-minimal window, which gtls_search reduces away.  Host pointers only
 * (opts->pointers_on_device => GTLS_EUNSUPPORTED); uses opts->dt0, device, stream and opts->path (1: the fused
 * small-N kernel of gtls_search's path = 1, with its limits; anything else: the general path); arrays must hold
 * ceil(n/stride) entries (n is always enough); *out_chi2_null (may be NULL) = chi2_0.  A window the kernel
 * never scored comes back as NaN.  Returns the number of starts (>= 1) or a negative error code. */
int64_t gtls_ring_window_chi2(const double* t, const double* y, const double* dy, int64_t n, double period,
                              double q, const double* tmpl, int32_t n_tmpl, const gtls_opts* opts,
                              int32_t* out_start, double* out_depth, double* out_dchi2, double* out_chi2_null);

/* Parity / debug export of steps a1-a2: phases (Eq. 10) and the stable phase-sort permutation
 * for each period.  out_phase [n_per*n] may be NULL; out_perm [n_per*n] (int32) is required.
 * out_phase[ip*n + i] is the phase of input point i; out_perm[ip*n + s] is the input index at
 * sorted position s. */
int gtls_fold_sort(const double* t, int64_t n, const double* periods, int64_t n_per,
                   const gtls_opts* opts, double* out_phase, int32_t* out_perm);

/* Parity / debug export of steps a3-a4 for ONE period: the gathered, wrap-padded prefix sums
 * (Eq. 14) of x1 = w r, x0 = w, x2 = w r^2 with w = 1/dy^2, r = 1 - y, in phase order.
 * Each output holds n + pad + 1 doubles, out[0] = 0, out[s+1] = sum of the first s+1 padded
 * entries (entries n..n+pad-1 repeat entries 0..pad-1, Fig. 3).  Any output may be NULL. */
int gtls_fold_scan(const double* t, const double* y, const double* dy, int64_t n, double period,
                   int64_t pad, const gtls_opts* opts, double* out_s1, double* out_s0,
                   double* out_s2);

/* Parity / debug export of steps a5-a7 for ONE (period, duration fraction q): for every strided
 * start k*stride < n writes the start index, the depth a, chi2_out = chi2_0 - (S2[s+D]-S2[s])
 * (Eq. 15 with the Eq. 11 edge term, reading G4) and chi2_in (Eq. 16).  Arrays must hold
 * ceil(n/stride) entries (n is always enough).  Returns the number of starts (>= 1) or a
 * negative error code. */
int64_t gtls_window_chi2(const double* t, const double* y, const double* dy, int64_t n,
                         double period, double q, const double* tmpl, int32_t n_tmpl,
                         const gtls_opts* opts, int32_t* out_start, double* out_depth,
                         double* out_chi2_out, double* out_chi2_in);

/* Step a9 alone: SR, SDE_raw, SDE and the summary indices from a chi2(P) array (used after a
 * period-sharded multi-GPU search has gathered chi2).  out_sde_raw / out_sde may be NULL.
 * Only the chi2 / SDE fields of out_summary are filled. */
int gtls_sde(const double* chi2, int64_t n_per, const gtls_opts* opts,
             double* out_sde_raw, double* out_sde, gtls_summary* out_summary);

/* ---- Trial grids built on the device (paper section 2.2) ------------------------------------------
 * Period grid: Ofir (2014) cubic frequency sampling, f_i = (A/3 i + C)^3, i = 1..N (Eq. 4)
 * with f_min = 2/S (Eq. 1), A of Eq. 5 (reading G21: its S is the time span in seconds, OS the
 * oversampling factor), C = f_min^(1/3) - A/3 and N = ceil(Eq. 6).  span and p_min in days, r_star and
 * m_star in solar units; p_min <= 0 takes f_max from the Roche limit (Eq. 3).  Periods come
 * out in days in ascending-frequency order (first = span/2, last ~ p_min).
 * gtls_period_grid_size returns N (>= 1) or a negative error code (GTLS_EINVAL: a parameter <= 0 or not
 * finite; GTLS_EGRID: f_max <= f_min, or N above 2^31).  gtls_period_grid writes out_periods[n_per]
 * (host or device per opts->pointers_on_device); n_per must equal gtls_period_grid_size(...). */
int64_t gtls_period_grid_size(double span, double r_star, double m_star, double oversampling, double p_min);
int gtls_period_grid(double span, double r_star, double m_star, double oversampling, double p_min,
                     const gtls_opts* opts, double* out_periods, int64_t n_per);

/* Duration grid: for every period n_dur fractions q = T14/P, log-spaced from min(k_min P^(-2/3), q_cap)
 * to min(k_max P^(-2/3), q_cap) with P in seconds (Eq. 8-9; cap PAPER.md:159; reading
 * G12).  GTLS defaults: k_min 20.05, k_max 620.84 s^(2/3), q_cap 0.15.  periods [n_per] in days (host or
 * device like the output), out_durations [n_per][n_dur] (the dur_per_period = 1 layout of gtls_search).
 * n_dur = 1 gives the lower edge.  GTLS_EINVAL: k_min <= 0, k_max < k_min, q_cap outside (0, 0.5];
 * GTLS_EGRID: a period <= 0 or not finite (its row is NaN). */
int gtls_duration_grid(const double* periods, int64_t n_per, int32_t n_dur, double k_min, double k_max,
                       double q_cap, const gtls_opts* opts, double* out_durations);

/* ---- Survey mode: many independent light curves in one call (BASELINE.json config 5) -----------------
 * Curve c is t/y/dy[curve_offset[c] .. curve_offset[c+1]) with its own period grid
 * period_grid[period_offset[c] .. period_offset[c+1]); duration_grid is [n_dur] shared by everything
 * (opts->dur_per_period = 0) or [period_offset[n_curves]][n_dur], rows in the order of period_grid
 * (dur_per_period = 1).  The offset arrays are HOST arrays of n_curves + 1 ascending entries starting at
 * 0; every other array is host or device per opts->pointers_on_device.  Outputs are concatenated in the
 * same order as period_grid: out_chi2 [total periods] (required), out_best / out_sde_raw / out_sde (may
 * be NULL); out_summary [n_curves] and out_status [n_curves] are HOST arrays and may be NULL.
 * Each curve is one gtls_search (same options, same results bit for bit) on an internal stream (ordered
 * after opts->stream at entry, joined before return).  GTLS_BATCH_LANES (environment, default 1, at most
 * 16) curves run concurrently, each lane on its own stream and host thread with its own slice of the
 * scratch: opts->workspace, when given, must hold gtls_batch_workspace_bytes(...).  The call returns
 * after all curves have finished.
 * Return: GTLS_OK when every curve returned GTLS_OK or GTLS_EDEGENERATE (see out_status), else the
 * error code of the first failing curve; curves after a failure are still searched. */
int gtls_search_batch(int32_t n_curves, const double* t, const double* y, const double* dy,
                      const int64_t* curve_offset, const double* period_grid,
                      const int64_t* period_offset, const double* duration_grid, int32_t n_dur,
                      const double* tmpl, int32_t n_tmpl, const gtls_opts* opts,
                      double* out_chi2, gtls_best* out_best, double* out_sde_raw, double* out_sde,
                      gtls_summary* out_summary, int32_t* out_status);
size_t gtls_batch_workspace_bytes(int32_t n_curves, const int64_t* curve_offset,
                                  const int64_t* period_offset, int32_t n_dur, const gtls_opts* opts);

/* Device scratch needed by gtls_search for these sizes and options (tile = opts->period_tile
 * or the automatic choice: enough for the worst case -- per-point errors, durations up to half a
 * period -- at its automatic tile, and for the common case -- one common error bar, durations up
 * to a fifth of a period -- at ITS larger automatic tile).  Pass a buffer of at least this size
 * in opts->workspace to avoid allocation inside the call. */
size_t gtls_workspace_bytes(int64_t n, int64_t n_per, int32_t n_dur, const gtls_opts* opts);

/* Device blocks the library allocates itself (the staged copies of host arrays, the scratch when
 * opts->workspace is NULL) are kept in a small pool between calls instead of being freed: at most four
 * free blocks of at most GTLS_CACHE_MB MiB each (environment, default 8192; 0 = no pool).  This call frees
 * them.  Caller-owned memory is never retained. */
void gtls_release_cache(void);

/* The search for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): the fused small-N path of gtls_search (opts->path = 1: fold, sort, pad, scans and
 * the chi2 rings of a period in one CTA's shared memory; then SR / SDE, Eq. 17) with ALL of
 * its scratch in one static device array of gtls_static_scratch_bytes() (~263 KB) that every GPU which loads
 * the library holds until exit.  It calls no cudaMalloc / cudaFree / allocating library routine and does not
 * use the block pool or opts->workspace.
 *   - Every array argument is a DEVICE pointer (opts->pointers_on_device is ignored); out_chi2, out_best,
 *     out_sde_raw and out_sde are all required ([n_per] each); out_summary (host) may be NULL.
 *   - Limits: 3 <= n <= GTLS_STATIC_MAX_N, n_dur <= 32, uniform dy, opts->top_k == 0, opts->chi2_fp32 == 0, and
 *     the limits of the fused kernel (window class strides <= 31 columns for this dt0, the folded arrays within
 *     one CTA's shared memory: n <= ~8000 for duration fractions up to 0.15).  Anything beyond returns
 *     GTLS_EUNSUPPORTED with the reason in gtls_last_cuda_error(): n, n_dur and the options before anything is
 *     launched, the rest after the two validation kernels (which is where dy and the durations are read).
 *   - Uses opts->dt0, dur_per_period, sde_kernel, device, stream.  Synchronises opts->stream (validation
 *     flags, summary), like gtls_search.  Results are those of gtls_search with path = 1, bit for bit.
 *   - The array is shared by ALL calls in the process on that GPU and keeps the previous call's contents (the
 *     call clears what must start at zero): calls that overlap on one GPU -- other threads, other streams --
 *     race on it.  Serialise them. */
#define GTLS_STATIC_MAX_N 8192
int gtls_search_static(const double* t, const double* y, const double* dy, int64_t n,
                       const double* period_grid, int64_t n_per, const double* duration_grid,
                       int32_t n_dur, const double* tmpl, int32_t n_tmpl, const gtls_opts* opts,
                       double* out_chi2, gtls_best* out_best, double* out_sde_raw, double* out_sde,
                       gtls_summary* out_summary);
size_t gtls_static_scratch_bytes(void);

/* Measurement aid (bench.py --peak-fp64), not part of the search: runs a register-only fp64 FMA kernel
 * (16 independent chains per thread, three distinct register operands per DFMA, 16 warps per SM) back to
 * back on opts->stream for about `seconds` (0 < seconds <= 60) of device time and returns the sustained
 * rate in TFLOP/s (2 flop per FMA lane) in *out_tflops; *out_ms (may be NULL) = device time measured with
 * CUDA events, *out_launches (may be NULL) = kernel launches timed.  This is the measured denominator
 * beside the derived fp64 peak of the chi2 stage's roofline ("measure it first
 * with a dependent-DFMA microbenchmark").  Uses opts->device and opts->stream only; synchronises. */
int gtls_peak_fp64(double seconds, const gtls_opts* opts, double* out_tflops, double* out_ms,
                   int64_t* out_launches);

const char* gtls_strerror(int code);
const char* gtls_version(void);
/* Text of the last CUDA error seen by the calling thread ("" if none). */
const char* gtls_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* GTLS_H_ */
