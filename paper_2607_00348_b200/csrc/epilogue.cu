// Step a9: chi2_min over the grid, SR(P) = chi2_min / chi2(P) (reading G15), its mean and
// population standard deviation (G16), SDE_raw (Eq. 17), the moving-median
// detrend with edge replication (G17/G18) and the argmax.
#include "gtls_internal.cuh"

namespace gtls {

namespace {

constexpr int kRedThreads = 1024;

__device__ __forceinline__ double block_sum(double v, double* s_buf) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();
    if (lane == 0) s_buf[warp] = v;
    __syncthreads();
    v = lane < (int)(blockDim.x >> 5) ? s_buf[lane] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;   // every thread of warp 0 holds the total; broadcast below
}

// One CTA: argmin (lowest index on ties), mean and population sigma of SR.  Fixed reduction
// shape => deterministic.
__global__ void __launch_bounds__(kRedThreads) k_sde_stats(const double* __restrict__ chi2,
                                                           long long n, SdeScratch* sc) {
    __shared__ double s_buf[32];
    __shared__ double s_val[32];
    __shared__ long long s_idx[32];
    __shared__ double s_bcast[2];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double mv = __longlong_as_double(0x7ff0000000000000LL);   // +inf
    long long mi = 0x7fffffffffffffffLL;
    for (long long i = threadIdx.x; i < n; i += blockDim.x) {
        const double c = chi2[i];
        if (c < mv || (c == mv && i < mi)) { mv = c; mi = i; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double ov = __shfl_xor_sync(0xffffffffu, mv, o);
        const long long oi = __shfl_xor_sync(0xffffffffu, mi, o);
        if (ov < mv || (ov == mv && oi < mi)) { mv = ov; mi = oi; }
    }
    if (lane == 0) { s_val[warp] = mv; s_idx[warp] = mi; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < (int)(blockDim.x >> 5); ++k)
            if (s_val[k] < mv || (s_val[k] == mv && s_idx[k] < mi)) { mv = s_val[k]; mi = s_idx[k]; }
        // no value compared below +inf (every chi2 is NaN or +inf): a degenerate spectrum whose argmin is
        // the first period, so that nothing downstream indexes with the sentinel
        if (mi == 0x7fffffffffffffffLL) { mi = 0; mv = __longlong_as_double(0x7ff8000000000000LL); }
        s_bcast[0] = mv;
        sc->chi2_min = mv; sc->argmin = mi;
    }
    __syncthreads();
    const double cmin = s_bcast[0];
    if (!(cmin > 0.0)) {
        if (threadIdx.x == 0) { sc->degenerate = 1; sc->mean_sr = 0.0; sc->sd_sr = 0.0; }
        return;
    }
    double acc = 0.0;
    for (long long i = threadIdx.x; i < n; i += blockDim.x) acc += __ddiv_rn(cmin, chi2[i]);
    acc = block_sum(acc, s_buf);
    if (threadIdx.x == 0) s_bcast[1] = __ddiv_rn(acc, (double)n);
    __syncthreads();
    const double mean = s_bcast[1];
    acc = 0.0;
    for (long long i = threadIdx.x; i < n; i += blockDim.x) {
        const double d = __ddiv_rn(cmin, chi2[i]) - mean;
        acc = fma(d, d, acc);
    }
    acc = block_sum(acc, s_buf);
    if (threadIdx.x == 0) {
        const double var = __ddiv_rn(acc, (double)n);
        sc->mean_sr = mean;
        sc->sd_sr = var > 0.0 ? sqrt(var) : 0.0;
        sc->degenerate = var > 0.0 ? 0 : 1;
    }
}

__global__ void __launch_bounds__(256) k_sde_raw(const double* __restrict__ chi2, long long n,
                                                 const SdeScratch* __restrict__ sc,
                                                 double* __restrict__ sde_raw) {
    const bool deg = sc->degenerate != 0;
    const double cmin = sc->chi2_min, mean = sc->mean_sr, sd = sc->sd_sr;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x)
        sde_raw[i] = deg ? 0.0 : __ddiv_rn(__ddiv_rn(cmin, chi2[i]) - mean, sd);
}

// order-preserving map double -> u64
__device__ __forceinline__ u64 ord(double x) {
    const u64 b = (u64)__double_as_longlong(x);
    return (b & 0x8000000000000000ull) ? ~b : (b | 0x8000000000000000ull);
}
__device__ __forceinline__ double unord(u64 k) {
    const u64 b = (k & 0x8000000000000000ull) ? (k & 0x7fffffffffffffffull) : ~k;
    return __longlong_as_double((long long)b);
}

// Median of the K-window around i (indices clamped = edge replication) by MSB-first radix
// select on the ordered bit pattern: 64 counting passes over the window, no local arrays.
__global__ void __launch_bounds__(128) k_sde_median(const double* __restrict__ sde_raw, long long n,
                                                    int kernel, const SdeScratch* __restrict__ sc,
                                                    double* __restrict__ sde) {
    const int h = (kernel - 1) / 2;
    const bool deg = sc->degenerate != 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x) {
        if (deg) { sde[i] = 0.0; continue; }
        if (kernel <= 1) { sde[i] = sde_raw[i]; continue; }
        u64 prefix = 0;
        for (int bit = 63; bit >= 0; --bit) {
            const u64 cand = prefix | (1ull << bit);
            int below = 0;
            for (int k = -h; k <= h; ++k) {
                long long j = i + k;
                j = j < 0 ? 0 : (j > n - 1 ? n - 1 : j);
                below += ord(sde_raw[j]) < cand ? 1 : 0;
            }
            if (below <= h) prefix = cand;      // the h-th order statistic is >= cand
        }
        sde[i] = sde_raw[i] - unord(prefix);
    }
}

// The same radix select with a warp per output (windows up to 32 * kMedPer values): every lane keeps
// its share of the window in registers as ordered bit patterns, a pass is kMedPer compares and one
// warp-wide add.  Same result bit for bit; ~60x lower latency than a thread per output.
constexpr int kMedPer = 8;
__global__ void __launch_bounds__(256) k_sde_median_warp(const double* __restrict__ sde_raw, long long n,
                                                         int kernel, const SdeScratch* __restrict__ sc,
                                                         double* __restrict__ sde) {
    const int h = (kernel - 1) / 2, lane = threadIdx.x & 31;
    const bool deg = sc->degenerate != 0;
    const long long warps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long i = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5; i < n; i += warps) {
        if (deg) { if (lane == 0) sde[i] = 0.0; continue; }
        u64 v[kMedPer];
#pragma unroll
        for (int e = 0; e < kMedPer; ++e) {
            const int k = e * 32 + lane;
            long long j = i - h + k;
            j = j < 0 ? 0 : (j > n - 1 ? n - 1 : j);
            v[e] = k < kernel ? ord(sde_raw[j]) : ~0ull;       // ~0: never below a candidate
        }
        u64 prefix = 0;
        for (int bit = 63; bit >= 0; --bit) {
            const u64 cand = prefix | (1ull << bit);
            int below = 0;
#pragma unroll
            for (int e = 0; e < kMedPer; ++e) below += v[e] < cand ? 1 : 0;
            below = __reduce_add_sync(0xffffffffu, below);
            if (below <= h) prefix = cand;                     // the h-th order statistic is >= cand
        }
        if (lane == 0) sde[i] = sde_raw[i] - unord(prefix);
    }
}

__global__ void __launch_bounds__(kRedThreads) k_sde_argmax(const double* __restrict__ sde,
                                                            const double* __restrict__ sde_raw,
                                                            long long n, SdeScratch* sc) {
    __shared__ double s_val[32];
    __shared__ long long s_idx[32];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double mv = __longlong_as_double((long long)0xfff0000000000000ULL);   // -inf
    long long mi = 0x7fffffffffffffffLL;
    for (long long i = threadIdx.x; i < n; i += blockDim.x) {
        const double c = sde[i];
        if (c > mv || (c == mv && i < mi)) { mv = c; mi = i; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double ov = __shfl_xor_sync(0xffffffffu, mv, o);
        const long long oi = __shfl_xor_sync(0xffffffffu, mi, o);
        if (ov > mv || (ov == mv && oi < mi)) { mv = ov; mi = oi; }
    }
    if (lane == 0) { s_val[warp] = mv; s_idx[warp] = mi; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < (int)(blockDim.x >> 5); ++k)
            if (s_val[k] > mv || (s_val[k] == mv && s_idx[k] < mi)) { mv = s_val[k]; mi = s_idx[k]; }
        if (sc->degenerate) { mi = sc->argmin; mv = 0.0; }
        sc->sde_max = mv; sc->sde_argmax = mi;
        sc->sde_raw_best = sde_raw[sc->argmin];
    }
}

// survey mode: the summary of every curve of a batch, one thread per curve
__global__ void __launch_bounds__(128) k_batch_summary(int n_curves, const long long* __restrict__ per_off,
                                                       const SdeScratch* __restrict__ sc, const gtls_best* __restrict__ best,
                                                       const double* __restrict__ periods, const CurveInfo* __restrict__ info,
                                                       const unsigned long long* __restrict__ counters, gtls_summary* out) {
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_curves) return;
    const long long p0 = per_off[c];
    const SdeScratch s = sc[c];
    const gtls_best b = best[p0 + s.argmin];
    gtls_summary o;
    o.best_period_idx = s.argmin;
    o.best_dur_idx = b.dur_idx;
    o.best_start = b.start;
    o.best_period = periods[p0 + s.argmin];
    o.best_t0 = b.t0;
    o.best_depth = b.depth;
    o.chi2_min = s.chi2_min;
    o.chi2_null = info[c].chi2_0;
    o.sde_raw_max = s.sde_raw_best;
    o.sde_max = s.sde_max;
    o.sde_argmax = s.sde_argmax;
    o.windows_evaluated = (int64_t)counters[2 * c];
    out[c] = o;
}

}  // namespace

void launch_batch_summary(int n_curves, const long long* per_off, const SdeScratch* sc, const gtls_best* best,
                          const double* periods, const CurveInfo* info, const unsigned long long* counters,
                          gtls_summary* out, cudaStream_t st) {
    k_batch_summary<<<(n_curves + 127) / 128, 128, 0, st>>>(n_curves, per_off, sc, best, periods, info, counters, out);
}

void launch_sde(const double* chi2, long long n_per, int kernel, double* sde_raw, double* sde,
                SdeScratch* scratch, cudaStream_t st, int* n_launches) {
    long long b = (n_per + 255) / 256;
    const int blocks = (int)(b > 148 * 16 ? 148 * 16 : b);
    long long bm = (n_per + 127) / 128;
    const int mblocks = (int)(bm > 148 * 64 ? 148 * 64 : bm);
    k_sde_stats<<<1, kRedThreads, 0, st>>>(chi2, n_per, scratch);
    k_sde_raw<<<blocks, 256, 0, st>>>(chi2, n_per, scratch, sde_raw);
    if (kernel > 1 && kernel <= 32 * kMedPer) {
        long long bw = (n_per + 7) / 8;                        // 8 warps per CTA, one output per warp and round
        const int wblocks = (int)(bw > 148 * 32 ? 148 * 32 : bw);
        k_sde_median_warp<<<wblocks, 256, 0, st>>>(sde_raw, n_per, kernel, scratch, sde);
    } else {
        k_sde_median<<<mblocks, 128, 0, st>>>(sde_raw, n_per, kernel, scratch, sde);
    }
    k_sde_argmax<<<1, kRedThreads, 0, st>>>(sde, sde_raw, n_per, scratch);
    if (n_launches) *n_launches += 4;
}

}  // namespace gtls
