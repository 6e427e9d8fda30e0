// Steps a5-a8 -- the per-period reduction (a8) and the per-window debug export.
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

// a8: per period, first strict minimum over ascending duration index.
__global__ void __launch_bounds__(128) k_reduce(TileArgs a, double* __restrict__ out_chi2,
                                                gtls_best* __restrict__ out_best,
                                                unsigned long long* __restrict__ counters) {
    const int pl = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long nwin = 0, npts = 0;
    if (pl < a.tile) {
        const Partial* pp = a.partial + (long long)pl * a.n_dur;
        const DurEntry* dd = a.durtab + (long long)pl * a.n_dur;
        int bj = -1;                 // no usable window at all: chi2_0, dur_idx 0, start 0 (reading G22)
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
            const int bs = bj >= 0 ? pp[bj].start : 0;
            b.dur_idx = bj >= 0 ? bj : 0; b.start = bs; b.depth = bj >= 0 ? pp[bj].depth : 0.0;
            const int mid = (bs + (dd[b.dur_idx].D - 1) / 2) % a.n;
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

void launch_reduce(const TileArgs& a, double* out_chi2, gtls_best* out_best,
                   unsigned long long* counters, cudaStream_t st) {
    k_reduce<<<(a.tile + 127) / 128, 128, 0, st>>>(a, out_chi2, out_best, counters);
}

void launch_window_export(const TileArgs& a, const double* s2, double q, int32_t* out_start,
                          double* out_depth, double* out_c_out, double* out_c_in, cudaStream_t st) {
    k_window_export<<<64, 256, 0, st>>>(a, s2, q, out_start, out_depth, out_c_out, out_c_in);
}

}  // namespace gtls
