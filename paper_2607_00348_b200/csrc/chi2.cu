// Steps a5-a8 -- general tiled path.
//   a5 depth:   rbar = (S1[s+D]-S1[s]) / (S0[s+D]-S0[s]),  a = max(rbar,0)/mean(g_D)   (Eq. 12-14)
//   a6 + a7:    chi2 = chi2_out + chi2_in = chi2_0 - 2 a C + a^2 G                     (Eq. 15-16)
//               C = sum_j g_D[j] x1[s+j],  G = sum_j g_D[j]^2 x0[s+j]
//               (the S2 = sum w r^2 window term of chi2_out, Eq. 15, cancels against the same
//               term inside chi2_in, Eq. 16, so the hot path never reads it; the debug export
//               gtls_window_chi2 evaluates both terms separately from S2.)
//   a8 reduce:  lexicographic argmin over (dchi2, dur_idx, start) per period.
#include <math_constants.h>

#include "gtls_internal.cuh"

namespace gtls {

namespace {

constexpr int kChiThreads = 256;
constexpr int kChiWarps = kChiThreads / 32;
constexpr int kJChunk = 4096;     // template points staged per pass
constexpr int kAccMax = 2048;     // window accumulators held in shared memory

struct Cand { double d; double depth; int s; int has; };

__device__ __forceinline__ void cand_offer(Cand& b, double d, int s, double depth) {
    if (!b.has || d < b.d || (d == b.d && s < b.s)) { b.d = d; b.s = s; b.depth = depth; b.has = 1; }
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

template <bool UNIFORM>
__global__ void __launch_bounds__(kChiThreads) k_chi2_v1(TileArgs a) {
    extern __shared__ double smem[];
    double* g = smem;                                   // [kJChunk]
    double* g2 = smem + kJChunk;                        // [kJChunk]   (!UNIFORM)
    double* accC = smem + (UNIFORM ? kJChunk : 2 * kJChunk);   // [kAccMax]
    double* accG = accC + kAccMax;                      // [kAccMax]   (!UNIFORM)
    __shared__ Cand s_best[kChiWarps];

    const int jd = blockIdx.x, pl = blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const DurEntry e = a.durtab[(long long)pl * a.n_dur + jd];
    Partial* out = a.partial + (long long)pl * a.n_dur + jd;
    if (e.skip) {
        if (threadIdx.x == 0) { out->valid = 0; out->dchi2 = 0.0; out->depth = 0.0; out->start = 0; }
        return;
    }
    const int D = e.D, stride = e.stride;
    const int nW = (a.n + stride - 1) / stride;
    const double* __restrict__ x1 = a.x1 + (long long)pl * a.pitch;
    const double* __restrict__ x0 = a.x0 + (long long)pl * a.pitch;
    const double* __restrict__ s1 = a.s1 + (long long)pl * a.spitch;
    const double* __restrict__ s0 = a.s0 + (long long)pl * a.spitch;
    const double w_u = a.w_uniform;
    const double G_u = w_u * e.gg2;
    const double sw_u = (double)D * w_u;
    Cand best; best.has = 0; best.d = 0.0; best.s = 0; best.depth = 0.0;

    for (int wbase = 0; wbase < nW; wbase += kAccMax) {
        const int wcnt = min(kAccMax, nW - wbase);
        for (int k = threadIdx.x; k < wcnt; k += kChiThreads) { accC[k] = 0.0; if (!UNIFORM) accG[k] = 0.0; }
        for (int j0 = 0; j0 < D; j0 += kJChunk) {
            const int jc = min(kJChunk, D - j0);
            __syncthreads();
            for (int j = threadIdx.x; j < jc; j += kChiThreads) {    // template -> shared memory
                const double gv = tmpl_at(a.tmpl, a.n_tmpl, j0 + j, D);
                g[j] = gv;
                if (!UNIFORM) g2[j] = gv * gv;
            }
            __syncthreads();
            if (D < 32) {
                // short windows: one thread per window (stride is 1..3, loads stay coalesced)
                for (int k = threadIdx.x; k < wcnt; k += kChiThreads) {
                    const double* p1 = x1 + (long long)(wbase + k) * stride + j0;
                    const double* p0 = x0 + (long long)(wbase + k) * stride + j0;
                    double c = 0.0, gg = 0.0;
                    for (int j = 0; j < jc; ++j) {
                        c = fma(g[j], p1[j], c);
                        if (!UNIFORM) gg = fma(g2[j], p0[j], gg);
                    }
                    accC[k] += c;
                    if (!UNIFORM) accG[k] += gg;
                }
            } else {
                // one warp per window, two windows in flight per warp
                for (int k = warp; k < wcnt; k += 2 * kChiWarps) {
                    const int kb = k + kChiWarps;
                    const bool two = kb < wcnt;
                    const double* pa1 = x1 + (long long)(wbase + k) * stride + j0;
                    const double* pb1 = x1 + (long long)(wbase + (two ? kb : k)) * stride + j0;
                    const double* pa0 = x0 + (long long)(wbase + k) * stride + j0;
                    const double* pb0 = x0 + (long long)(wbase + (two ? kb : k)) * stride + j0;
                    double ca = 0.0, cb = 0.0, ga = 0.0, gb = 0.0;
#pragma unroll 4
                    for (int j = lane; j < jc; j += 32) {
                        const double gv = g[j];
                        ca = fma(gv, pa1[j], ca);
                        cb = fma(gv, pb1[j], cb);
                        if (!UNIFORM) {
                            const double g2v = g2[j];
                            ga = fma(g2v, pa0[j], ga);
                            gb = fma(g2v, pb0[j], gb);
                        }
                    }
                    ca = warp_sum(ca); cb = warp_sum(cb);
                    if (!UNIFORM) { ga = warp_sum(ga); gb = warp_sum(gb); }
                    if (lane == 0) {
                        accC[k] += ca;
                        if (!UNIFORM) accG[k] += ga;
                        if (two) { accC[kb] += cb; if (!UNIFORM) accG[kb] += gb; }
                    }
                }
            }
        }
        __syncthreads();
        for (int k = threadIdx.x; k < wcnt; k += kChiThreads) {      // a5 + a8 per window
            const int s = (wbase + k) * stride;
            const double swr = s1[s + D] - s1[s];
            const double sw = UNIFORM ? sw_u : s0[s + D] - s0[s];
            const double rbar = __ddiv_rn(swr, sw);
            const double depth = __ddiv_rn(fmax(rbar, 0.0), e.gbar);
            const double C = accC[k];
            const double G = UNIFORM ? G_u : accG[k];
            const double d = -2.0 * depth * C + (depth * depth) * G;
            cand_offer(best, d, s, depth);
        }
        __syncthreads();
    }
    // CTA-wide lexicographic min on (d, s)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        Cand c;
        c.d = __shfl_xor_sync(0xffffffffu, best.d, o);
        c.depth = __shfl_xor_sync(0xffffffffu, best.depth, o);
        c.s = __shfl_xor_sync(0xffffffffu, best.s, o);
        c.has = __shfl_xor_sync(0xffffffffu, best.has, o);
        if (c.has) cand_offer(best, c.d, c.s, c.depth);
    }
    if (lane == 0) s_best[warp] = best;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < kChiWarps; ++k)
            if (s_best[k].has) cand_offer(best, s_best[k].d, s_best[k].s, s_best[k].depth);
        out->valid = best.has; out->dchi2 = best.d; out->depth = best.depth; out->start = best.s;
    }
}

// a8: per period, first strict minimum over ascending duration index.
__global__ void __launch_bounds__(128) k_reduce(TileArgs a, double* __restrict__ out_chi2,
                                                gtls_best* __restrict__ out_best,
                                                unsigned long long* __restrict__ counters) {
    const int pl = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long nwin = 0, npts = 0;
    if (pl < a.tile) {
        const Partial* pp = a.partial + (long long)pl * a.n_dur;
        const DurEntry* dd = a.durtab + (long long)pl * a.n_dur;
        int bj = -1;
        double bd = 0.0;
        for (int jd = 0; jd < a.n_dur; ++jd) {
            unsigned long long nw = (unsigned long long)((a.n + dd[jd].stride - 1) / dd[jd].stride);
            if (a.top_k > 0 && nw > (unsigned long long)a.top_k) nw = (unsigned long long)a.top_k;   // pruning variant
            nwin += nw;
            if (!dd[jd].skip) npts += nw * (unsigned long long)dd[jd].D;
            if (!pp[jd].valid) continue;
            if (bj < 0 || pp[jd].dchi2 < bd) { bj = jd; bd = pp[jd].dchi2; }
        }
        out_chi2[a.p0 + pl] = *a.chi2_0 + bd;
        if (out_best) {
            gtls_best b;
            b.dur_idx = bj; b.start = pp[bj].start; b.depth = pp[bj].depth;
            const int mid = (pp[bj].start + (dd[bj].D - 1) / 2) % a.n;
            const u32 src = a.perm[(long long)pl * a.n + mid];
            b.t0 = a.t[src < (u32)a.n ? src : 0u];      // (a tile whose bucket sort overflowed is recomputed)
            out_best[a.p0 + pl] = b;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        nwin += __shfl_xor_sync(0xffffffffu, nwin, o);
        npts += __shfl_xor_sync(0xffffffffu, npts, o);
    }
    if ((threadIdx.x & 31) == 0 && counters) { atomicAdd(&counters[0], nwin); atomicAdd(&counters[1], npts); }
}

// Debug export: every strided window of one (period, q), both chi2 terms kept separate.
__global__ void __launch_bounds__(256) k_window_export(TileArgs a, const double* __restrict__ s2,
                                                       double q, int32_t* out_start,
                                                       double* out_depth, double* out_c_out,
                                                       double* out_c_in) {
    const int D = points_in_duration(q, a.n);
    const int stride = t0_stride(D, a.dt0);
    const int nW = (a.n + stride - 1) / stride;
    // mean(g_D) with a sequential sum per thread (tiny problem sizes only)
    double sg = 0.0;
    for (int j = 0; j < D; ++j) sg += tmpl_at(a.tmpl, a.n_tmpl, j, D);
    const double gbar = __ddiv_rn(sg, (double)D);
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < nW; k += gridDim.x * blockDim.x) {
        const int s = k * stride;
        const double swr = a.s1[s + D] - a.s1[s];
        const double sw = a.s0[s + D] - a.s0[s];
        const double swr2 = s2[s + D] - s2[s];
        const double depth = __ddiv_rn(fmax(__ddiv_rn(swr, sw), 0.0), gbar);
        double C = 0.0, G = 0.0;
        for (int j = 0; j < D; ++j) {
            const double gv = tmpl_at(a.tmpl, a.n_tmpl, j, D);
            C = fma(gv, a.x1[s + j], C);
            G = fma(gv * gv, a.x0[s + j], G);
        }
        out_start[k] = s;
        out_depth[k] = depth;
        out_c_out[k] = *a.chi2_0 - swr2;                                   // a6 (Eq. 15 - Eq. 11)
        out_c_in[k] = swr2 - 2.0 * depth * C + (depth * depth) * G;        // a7 (Eq. 16)
    }
}

}  // namespace

void launch_chi2(const TileArgs& a, cudaStream_t st) {
    const dim3 grid(a.n_dur, a.tile);
    if (a.uniform) {
        const size_t sm = (size_t)(kJChunk + kAccMax) * sizeof(double);
        static bool set = false;
        if (!set) { cudaFuncSetAttribute(k_chi2_v1<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm); set = true; }
        k_chi2_v1<true><<<grid, kChiThreads, sm, st>>>(a);
    } else {
        const size_t sm = (size_t)(2 * kJChunk + 2 * kAccMax) * sizeof(double);
        static bool set = false;
        if (!set) { cudaFuncSetAttribute(k_chi2_v1<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm); set = true; }
        k_chi2_v1<false><<<grid, kChiThreads, sm, st>>>(a);
    }
}

void launch_reduce(const TileArgs& a, double* out_chi2, gtls_best* out_best,
                   unsigned long long* counters, cudaStream_t st) {
    k_reduce<<<(a.tile + 127) / 128, 128, 0, st>>>(a, out_chi2, out_best, counters);
}

void launch_window_export(const TileArgs& a, const double* s2, double q, int32_t* out_start,
                          double* out_depth, double* out_c_out, double* out_c_in, cudaStream_t st) {
    k_window_export<<<64, 256, 0, st>>>(a, s2, q, out_start, out_depth, out_c_out, out_c_in);
}

}  // namespace gtls
