// Internal declarations shared by the libgtls translation units (sm_100a only).
// Not part of the ABI; see include/gtls.h for the boundary.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "gtls.h"

namespace gtls {

typedef unsigned long long u64;
typedef unsigned int u32;

// One (period, duration) trial, step a5 prerequisites.
struct DurEntry {
    int32_t D;        // points per duration: clamp(floor(q*n), 1, n-1)      (G11)
    int32_t stride;   // max(1, floor(D*dt0))                                (Eq. 18, G9)
    double  gbar;     // mean of the resampled template g_D                  (Eq. 12-13, G5/G6)
    double  gg2;      // sum_j g_D[j]^2  (G = w * gg2 when dy is uniform)
    int32_t skip;     // 1 when an earlier duration index of this period has the same D
    int32_t pad_;
};

// Per-(period, duration) partial result of the window scan (a8 input).
struct Partial {
    double  dchi2;    // chi2 - chi2_0 of the best window of this trial
    double  depth;
    int32_t start;
    int32_t valid;
};

// Flags and scalars produced by the a0 kernels and read back once by the host.
struct CurveInfo {
    double chi2_0;        // sum_i w_i r_i^2
    double w_min, w_max;  // uniform-dy detection
    double q_max;         // largest duration fraction in the grid
    int32_t bad_curve;    // count of non-finite t/y/dy or dy <= 0
    int32_t bad_period;   // count of non-finite or <= 0 periods
    int32_t bad_duration; // count of fractions outside (0, 0.5]
    int32_t pad_;
};

// chi2 ring kernel variants: ring size index (0..5 = 24, 21, 16, 12, 8, 4 taps) + 6 * narrow
constexpr int kChi2Rings = 6;
constexpr int kChi2Variants = 2 * kChi2Rings;
constexpr int kBinBlocks = 148;      // CTAs of k_bin_trials; trial_count holds kChi2Variants * (1 + kBinBlocks) ints
constexpr int kXMargin = 40;         // zeroed doubles behind every period's wrap pad in x1 / x0 (k_durtab; read by the ring kernels' row copies)
constexpr int kChi2NarrowMax = 16;   // largest class stride handled by the narrow variants
// Window classes of a trial with M = ceil(D/stride) taps: the smallest count that leaves at most 24 taps
// per class when the class stride stays narrow (<= kChi2NarrowMax), at most 21 otherwise and when the
// stride is 1 (32 side-by-side segments of a 24-ring do not fit the window table).  The 24-ring is a
// narrow-path ring only: as a wide kernel it is slower per tap than the pipelined 21-ring (measured on
// c3 at dt0 = 0.01).  (A 28-ring was measured too: its unrolled body outgrows the instruction cache.)
// dy not uniform: the narrow path carries two rings (C and G) per lane, so its rings hold at most 16 taps
// (8 when the stride is 1: 32 segments x two tables); strides above 16 use the wide 21-ring.
__host__ __device__ __forceinline__ int chi2_classes(int M, int stride, bool uniform) {
    if (uniform) {
        if (stride == 1) return (M + 20) / 21;
        const int c = (M + 23) / 24;
        return c * stride <= kChi2NarrowMax ? c : (M + 20) / 21;
    }
    if (stride > kChi2NarrowMax) return (M + 20) / 21;
    int c = (M + 15) / 16;                             // a class stride of 17 .. 32 is a wide march with
    if (stride == 1 && M > 8 && c < 2) c = 2;          // twice the lanes a single class would fill
    return c;                                          // (stride 1 with one class: at most 8 taps)
}
__host__ __device__ __forceinline__ int chi2_ring_index(int taps) {
    return taps > 21 ? 0 : (taps > 16 ? 1 : (taps > 12 ? 2 : (taps > 8 ? 3 : (taps > 4 ? 4 : 5))));
}

// bucket sort (bucket_sort.cu)
constexpr int kMaxBuckets = 2048;     // buckets per period (power of two)
#ifndef GTLS_BUCKET_TARGET
#define GTLS_BUCKET_TARGET 280
#define GTLS_BUCKET_CAP 384
#endif
constexpr int kBucketTarget = GTLS_BUCKET_TARGET;   // aimed-at mean bucket size
constexpr int kBucketCap = GTLS_BUCKET_CAP;      // largest bucket the shared-memory sort takes; beyond: LSD fallback

constexpr int kRadixThreads = 256;
constexpr int kRadixItems = 8;
constexpr int kRadixTile = kRadixThreads * kRadixItems;   // 2048 keys per CTA
constexpr int kRadixWarps = kRadixThreads / 32;

// ---- phase / template arithmetic shared by kernels -------------------------------------
// Eq. 10: one IEEE fp64 division, floor, exact subtraction.  No reciprocal
// multiply and no fast-math anywhere in this library, so phases are bit-identical to any
// IEEE-754 host evaluation of the same expression.
__device__ __forceinline__ double fold_phase(double t, double period) {
    const double q = __ddiv_rn(t, period);
    return q - floor(q);
}

// Sortable key: floor(phase * 2^32) is a monotone (non-strict) map of the phase, so ordering
// by (key32, full phase, index) equals ordering by (phase, index).  The rare equal-key runs
// are re-ordered by the full fp64 phase in the tie fix-up kernel.
__device__ __forceinline__ u32 phase_key32(double phase) {
    const double s = phase * 4294967296.0;
    return s >= 4294967295.0 ? 0xFFFFFFFFu : (u32)(u64)s;
}

// Template deficit resampled to D points by linear interpolation at cell centres (G14).
__device__ __forceinline__ double tmpl_at(const double* __restrict__ tmpl, int n_tmpl, int j, int D) {
    const double u = __ddiv_rn((double)j + 0.5, (double)D) * (double)(n_tmpl - 1);
    int k = (int)floor(u);
    k = k > n_tmpl - 2 ? n_tmpl - 2 : k;
    k = k < 0 ? 0 : k;
    const double frac = u - (double)k;
    const double a = tmpl[k];
    return a + frac * (tmpl[k + 1] - a);
}

__device__ __forceinline__ int points_in_duration(double q, int n) {
    double d = floor(q * (double)n);
    d = d < 1.0 ? 1.0 : d;
    d = d > (double)(n - 1) ? (double)(n - 1) : d;
    return (int)d;
}

__device__ __forceinline__ int t0_stride(int D, double dt0) {
    if (!(dt0 > 0.0)) return 1;
    const double s = floor((double)D * dt0);
    return s < 1.0 ? 1 : (int)s;
}

// LSD path: segments (periods of the tile) a kernel has to process
__device__ __forceinline__ int seg_count(const int* list, const int* count, int tile) { return list ? *count : tile; }
__device__ __forceinline__ int seg_at(const int* list, int s) { return list ? list[s] : s; }

// ---- host-side launchers (one per kernel family) ----------------------------------------
struct TileArgs {
    int n;                 // points in the light curve
    int n_dur;
    int n_tmpl;
    int tile;              // periods in this tile
    long long p0;          // index of the first period of the tile
    int dur_per_period;
    double dt0;
    int uniform;           // all dy equal
    double w_uniform;      // the common weight when uniform
    int pitch;             // doubles per period in x1/x0 (>= n + Dmax)
    int spitch;            // doubles per period in S1/S0 (= pitch + 1 rounded up)
    const double* t;       // [n]
    const double* wr;      // [n]  w_i r_i
    const double* w;       // [n]  w_i
    const double* wr2;     // [n]  w_i r_i^2 (debug exports only)
    const double* periods; // [n_per]
    const double* durs;    // duration grid
    const double* tmpl;    // [n_tmpl]
    const double* chi2_0;  // device scalar (CurveInfo::chi2_0)
    u64* keys_a;           // [tile*n]
    u64* keys_b;           // [tile*n]
    u32* counts;           // [tile*256*nt]
    DurEntry* durtab;      // [tile*n_dur]
    double* x1; double* x0;   // [tile*pitch]
    double* s1; double* s0;   // [tile*spitch]
    Partial* partial;      // [tile*n_dur]
    u32* perm;             // [tile*n]   sorted position -> input index
    const int* seg_list;   // LSD path: periods (tile-local) to process, or nullptr = all of the tile
    const int* seg_count;  // number of entries of seg_list (device)
    int* trial_list;       // [kChi2Variants][tile*n_dur] trial indices binned by chi2 kernel variant
    int* trial_count;      // [kChi2Variants] totals + [kBinBlocks][kChi2Variants] per-CTA counts + [kChi2Variants] trial queues
    int top_k;             // > 0: chi2 only at the K deepest starts of every trial (chi2_topk.cu, reading G19)
    int chi2_fp32;         // 1: fp32 ring arithmetic in the chi2 kernels (gtls_opts.chi2_fp32)
    const double* gtab;    // [2*(gtab_max+1)] sum g_D, sum g_D^2 for D = 1 .. gtab_max (k_gtab)
    int gtab_max;
    double* dbg_dchi2;     // debug export only (gtls_ring_window_chi2): per-window dchi2 / depth written by the ring
    double* dbg_depth;     // kernels' scoring, indexed by start / stride; nullptr in every search
};

// Arguments of the fused fold / bucket sort / gather / scan fast path (bucket_sort.cu).
struct BucketArgs {
    int n, tile, nbk, shift;   // points, periods in the tile, buckets per period, 32 - log2(nbk)
    int ncta;                  // count / scatter CTAs per period (bucket_cta_count(n))
    long long p0;
    int n_dur, pad_override;   // pad = max D of the period's durtab row unless pad_override >= 0
    int pitch, spitch;
    const double* t; const double* wr; const double* w; const double* wr2;
    const double* periods;
    const DurEntry* durtab;
    unsigned short* hist;      // [tile*ncta*nbk] keys of every count CTA per bucket
    u32* start;                // [tile*(nbk+1)]
    u32* rel;                  // [tile*ncta*nbk] where a CTA's keys start inside the bucket
    int* fb_flag;              // [tile] 1: a bucket of this period exceeded kBucketCap (LSD path takes it)
    int* fb_list;              // [tile] those periods, any order
    int* fb_count;             // [1]
    u64* keys;                 // [tile*n] bucketed keys
    u32* perm;                 // [tile*n]
    double* x1; double* s1; double* x0; double* s0; double* x2; double* s2;
};
int bucket_count_for(int n);
int bucket_cta_count(int n);
// count + bucket starts + fallback list; then (after the caller forked the fallback path) scatter + sort + prefix / pad
void launch_bucket_sort_head(const BucketArgs& b, cudaStream_t st);
void launch_bucket_sort_tail(const BucketArgs& b, bool has0, bool has2, bool sort_only, cudaStream_t st);

// A high-priority side stream with a fork and a join event, per host thread, bound to the device of the
// thread's first call.  which: 0 = chi2 variants, 1 = LSD fallback of the sort.  nullptr when streams
// are switched off (GTLS_STREAMS=0), creation failed, or the current device is another one: the caller then
// launches everything on its own stream.
struct SideStream { cudaStream_t s; cudaEvent_t fork, join; };
SideStream* side_stream(int which);

void launch_curve_pre(const double* t, const double* y, const double* dy, int n, double* wr,
                      double* w, double* wr2, CurveInfo* info, cudaStream_t st);
// survey mode (api_batch.cu): per-curve arrays + validation flags for every curve of a concatenated batch
void launch_batch_pre(int n_curves, const double* t, const double* y, const double* dy, const long long* curve_off,
                      const double* periods, const long long* per_off, const double* durs, int n_dur,
                      int dur_per_period, double* wr, double* w, double* wr2, CurveInfo* info, cudaStream_t st);
void launch_grid_check(const double* periods, long long n_per, const double* durs,
                       long long n_durs_total, CurveInfo* info, cudaStream_t st);
constexpr int kTopKMax = 8;   // largest gtls_opts.top_k the pruning kernel takes (per-lane lists live in registers)
void launch_chi2_topk(const TileArgs& a, cudaStream_t st);
void launch_gtab(const double* tmpl, int n_tmpl, int gtab_max, double* gtab, cudaStream_t st);
void launch_durtab(const TileArgs& a, cudaStream_t st);
// grids.cu: Eq. 4 period grid from the host-side constants A/3 and C; Eq. 8-9 duration fractions
void launch_period_grid(double a3, double c, long long n_per, double* out, cudaStream_t st);
void launch_duration_grid(const double* periods, long long n_per, int n_dur, double k_min, double k_max,
                          double q_cap, double* out, int* bad, cudaStream_t st);
// bins the tile's trials by chi2 kernel variant (order preserved); skipped trials get an invalid Partial
void launch_bin_trials(const TileArgs& a, cudaStream_t st);
void launch_fold_keys(const TileArgs& a, double* phase_out, cudaStream_t st);
// sorts keys_a (in place semantics: result is returned in the pointer the function returns)
u64* launch_phase_sort(const TileArgs& a, cudaStream_t st, int* n_launches);
void launch_gather_scan(const TileArgs& a, const u64* sorted, double* x2, double* s2,
                        int pad_override, cudaStream_t st);
void launch_chi2_ring(const TileArgs& a, cudaStream_t st);   // register-ring correlation kernel (default)
// counters[0] += windows of all trials, counters[1] += sum of D over evaluated windows
void launch_reduce(const TileArgs& a, double* out_chi2, gtls_best* out_best,
                   unsigned long long* counters, cudaStream_t st);
void launch_window_export(const TileArgs& a, const double* s2, double q, int32_t* out_start,
                          double* out_depth, double* out_c_out, double* out_c_in, cudaStream_t st);
void launch_perm_export(const TileArgs& a, const u64* sorted, int32_t* out_perm, cudaStream_t st);

void launch_topk_sde(const double* sde, long long n, int K, unsigned char* mark, long long* sel, cudaStream_t st);
void launch_gather_refine(const double* periods, const double* durs, int dur_per_period, int n_dur,
                          const long long* sel, int K, double* per2, double* dur2, cudaStream_t st);
void launch_merge_refined(const long long* sel, int K, const double* chi2b, const gtls_best* bestb, double* chi2,
                          gtls_best* best, cudaStream_t st);

// Fused small-N path (small.cu): a batch of light curves, one work item per (curve, period).
struct SmallArgs {
    long long n_items;            // total periods over all curves
    int n_dur, n_tmpl, dur_per_period;
    double dt0;
    const long long* curve_off;   // device [n_curves + 1]: offsets of the curves in t / wr
    const long long* per_off;     // device [n_curves + 1]: offsets of the curves in periods / outputs
    const double* t;              // concatenated light-curve times
    const double* wr;             // concatenated w_i r_i
    const CurveInfo* info;        // [n_curves]: chi2_0, the common weight (w_min)
    const double* periods;        // [n_items]
    const double* durs;           // [n_dur] or [n_items][n_dur]
    const double* tmpl;
    const double* gtab;           // sum g_D, sum g_D^2 for every D the grids can ask for
    double* out_chi2;             // [n_items]
    gtls_best* out_best;          // [n_items] or nullptr
    unsigned long long* counters; // [n_curves][2]: windows, window points
    unsigned long long* queue;    // work counter (zeroed by the caller)
    int xs_len, n_max;            // set by launch_tls_small
    double* dbg_dchi2;            // debug export only (gtls_ring_window_chi2, path = 1): per-window dchi2 / depth of a
    double* dbg_depth;            // one-curve, one-period, one-duration call, indexed by start / stride; nullptr otherwise
};
size_t small_smem_bytes(int n_max, int d_max);
// dy uniform is the caller's check; this one covers sizes: shared memory, n_dur, class strides <= 31
bool small_path_fits(int n_max, int d_max, int n_dur, double dt0);
int launch_tls_small(SmallArgs& a, int n_max, int d_max, int sm_count, cudaStream_t st);   // returns a cudaError_t

struct SdeScratch {      // device scalars of the epilogue
    double chi2_min, mean_sr, sd_sr, sde_raw_best, sde_max;
    long long argmin, sde_argmax;
    int degenerate, pad_;
};
// one gtls_summary per curve of a batch from the epilogue scalars, the best records and the window counters
void launch_batch_summary(int n_curves, const long long* per_off, const SdeScratch* sc, const gtls_best* best,
                          const double* periods, const CurveInfo* info, const unsigned long long* counters,
                          gtls_summary* out, cudaStream_t st);
void launch_sde(const double* chi2, long long n_per, int kernel, double* sde_raw, double* sde,
                SdeScratch* scratch, cudaStream_t st, int* n_launches);

}  // namespace gtls
