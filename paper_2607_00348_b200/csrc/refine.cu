// Two-stage hierarchical search (section 2.5): helpers of gtls_search_two_stage.
//   k_topk_sde      the n_refine trial periods of highest SDE after the coarse stage (ties -> lower index)
//   k_gather_refine their periods and duration rows, packed for the stride-1 second stage
//   k_merge_refined the refined chi2 / best records replace the coarse ones
#include "gtls_internal.cuh"

namespace gtls {

namespace {

// One CTA; K rounds of a block-wide argmax over the not yet selected entries.  K is ~200 and n_per a few
// 1e5, so this is ~1e8 loads: a few milliseconds, once per search.
__global__ void __launch_bounds__(1024) k_topk_sde(const double* __restrict__ sde, long long n, int K,
                                                   unsigned char* __restrict__ mark, long long* __restrict__ sel) {
    __shared__ double s_val[32];
    __shared__ long long s_idx[32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (long long i = threadIdx.x; i < n; i += blockDim.x) mark[i] = 0;
    __syncthreads();
    for (int k = 0; k < K; ++k) {
        double mv = __longlong_as_double((long long)0xfff0000000000000ULL);   // -inf
        long long mi = 0x7fffffffffffffffLL;
        for (long long i = threadIdx.x; i < n; i += blockDim.x) {
            if (mark[i]) continue;
            const double v = sde[i];
            if (v > mv || (v == mv && i < mi) || mi == 0x7fffffffffffffffLL) { mv = v; mi = i; }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double ov = __shfl_xor_sync(0xffffffffu, mv, o);
            const long long oi = __shfl_xor_sync(0xffffffffu, mi, o);
            if (oi != 0x7fffffffffffffffLL && (mi == 0x7fffffffffffffffLL || ov > mv || (ov == mv && oi < mi))) { mv = ov; mi = oi; }
        }
        if (lane == 0) { s_val[warp] = mv; s_idx[warp] = mi; }
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int w = 1; w < (int)(blockDim.x >> 5); ++w) {
                const double ov = s_val[w];
                const long long oi = s_idx[w];
                if (oi != 0x7fffffffffffffffLL && (mi == 0x7fffffffffffffffLL || ov > mv || (ov == mv && oi < mi))) { mv = ov; mi = oi; }
            }
            sel[k] = mi;
            mark[mi] = 1;
        }
        __syncthreads();
    }
}

__global__ void __launch_bounds__(256) k_gather_refine(const double* __restrict__ periods,
                                                       const double* __restrict__ durs, int dur_per_period,
                                                       int n_dur, const long long* __restrict__ sel, int K,
                                                       double* __restrict__ per2, double* __restrict__ dur2) {
    for (int g = blockIdx.x * blockDim.x + threadIdx.x; g < K * n_dur; g += gridDim.x * blockDim.x) {
        const int k = g / n_dur, jd = g - k * n_dur;
        const long long ip = sel[k];
        if (jd == 0) per2[k] = periods[ip];
        dur2[g] = dur_per_period ? durs[ip * n_dur + jd] : durs[jd];
    }
}

__global__ void __launch_bounds__(256) k_merge_refined(const long long* __restrict__ sel, int K,
                                                       const double* __restrict__ chi2b,
                                                       const gtls_best* __restrict__ bestb,
                                                       double* __restrict__ chi2, gtls_best* __restrict__ best) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= K) return;
    const long long ip = sel[k];
    chi2[ip] = chi2b[k];
    if (best) best[ip] = bestb[k];
}

}  // namespace

void launch_topk_sde(const double* sde, long long n, int K, unsigned char* mark, long long* sel, cudaStream_t st) {
    k_topk_sde<<<1, 1024, 0, st>>>(sde, n, K, mark, sel);
}
void launch_gather_refine(const double* periods, const double* durs, int dur_per_period, int n_dur,
                          const long long* sel, int K, double* per2, double* dur2, cudaStream_t st) {
    const int total = K * n_dur;
    k_gather_refine<<<(total + 255) / 256, 256, 0, st>>>(periods, durs, dur_per_period, n_dur, sel, K, per2, dur2);
}
void launch_merge_refined(const long long* sel, int K, const double* chi2b, const gtls_best* bestb, double* chi2,
                          gtls_best* best, cudaStream_t st) {
    k_merge_refined<<<(K + 255) / 256, 256, 0, st>>>(sel, K, chi2b, bestb, chi2, best);
}

}  // namespace gtls
