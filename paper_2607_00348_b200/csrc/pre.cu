// Step a0: per-curve arrays (w, w r, w r^2, chi2_0), input validation, and the per-tile
// duration table (D, stride, mean(g_D), sum g_D^2) -- SURVEY 8(a) row a0, 8(c) step 3.
#include "gtls_internal.cuh"

namespace gtls {

namespace {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// One CTA of 1024 threads: deterministic strided accumulation + fixed-shape tree.
__device__ __forceinline__ void curve_pre_body(const double* __restrict__ t,
                                               const double* __restrict__ y,
                                               const double* __restrict__ dy, int n,
                                               double* __restrict__ wr, double* __restrict__ w,
                                               double* __restrict__ wr2, CurveInfo* info) {
    __shared__ double s_sum[32], s_min[32], s_max[32];
    __shared__ int s_bad[32];
    double acc = 0.0, wmin = 1e300, wmax = 0.0;
    int bad = 0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const double ti = t[i], yi = y[i], di = dy[i];
        const double wi = __ddiv_rn(1.0, di * di);     // w_i = 1/dy_i^2
        const double ri = 1.0 - yi;                    // flux deficit (model == 1)
        const double wri = wi * ri;
        const double wr2i = wri * ri;
        // dy so small that dy^2 underflows gives w = inf and w r = NaN: rejected like a non-finite input
        const bool ok = isfinite(ti) && isfinite(yi) && isfinite(di) && di > 0.0 && isfinite(wi) && isfinite(wri) &&
                        isfinite(wr2i);
        bad += ok ? 0 : 1;
        w[i] = wi; wr[i] = wri; wr2[i] = wr2i;
        acc += wr2i;
        wmin = fmin(wmin, wi); wmax = fmax(wmax, wi);
    }
    acc = warp_sum(acc);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        wmin = fmin(wmin, __shfl_xor_sync(0xffffffffu, wmin, o));
        wmax = fmax(wmax, __shfl_xor_sync(0xffffffffu, wmax, o));
        bad += __shfl_xor_sync(0xffffffffu, bad, o);
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { s_sum[warp] = acc; s_min[warp] = wmin; s_max[warp] = wmax; s_bad[warp] = bad; }
    __syncthreads();
    if (warp == 0) {
        const int nw = blockDim.x >> 5;
        acc = lane < nw ? s_sum[lane] : 0.0;
        wmin = lane < nw ? s_min[lane] : 1e300;
        wmax = lane < nw ? s_max[lane] : 0.0;
        bad = lane < nw ? s_bad[lane] : 0;
        acc = warp_sum(acc);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            wmin = fmin(wmin, __shfl_xor_sync(0xffffffffu, wmin, o));
            wmax = fmax(wmax, __shfl_xor_sync(0xffffffffu, wmax, o));
            bad += __shfl_xor_sync(0xffffffffu, bad, o);
        }
        if (lane == 0) {
            info->chi2_0 = acc; info->w_min = wmin; info->w_max = wmax; info->bad_curve = bad;
        }
    }
}

__global__ void __launch_bounds__(1024) k_curve_pre(const double* __restrict__ t, const double* __restrict__ y,
                                                    const double* __restrict__ dy, int n, double* __restrict__ wr,
                                                    double* __restrict__ w, double* __restrict__ wr2, CurveInfo* info) {
    curve_pre_body(t, y, dy, n, wr, w, wr2, info);
}
// survey mode: one CTA per light curve of the concatenated batch
__global__ void __launch_bounds__(1024) k_curve_pre_batch(const double* __restrict__ t, const double* __restrict__ y,
                                                          const double* __restrict__ dy, const long long* __restrict__ curve_off,
                                                          double* __restrict__ wr, double* __restrict__ w,
                                                          double* __restrict__ wr2, CurveInfo* info) {
    const long long c0 = curve_off[blockIdx.x];
    curve_pre_body(t + c0, y + c0, dy + c0, (int)(curve_off[blockIdx.x + 1] - c0), wr + c0, w + c0, wr2 + c0,
                   info + blockIdx.x);
}

// Many CTAs; integer counters and the max are order independent, so atomics keep it exact.
__global__ void __launch_bounds__(256) k_grid_check(const double* __restrict__ periods,
                                                    long long n_per,
                                                    const double* __restrict__ durs,
                                                    long long n_durs, CurveInfo* info) {
    int bp = 0, bd = 0;
    double qmax = 0.0;
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long nth = (long long)gridDim.x * blockDim.x;
    for (long long i = tid; i < n_per; i += nth) {
        const double p = periods[i];
        bp += (isfinite(p) && p > 0.0) ? 0 : 1;
    }
    for (long long i = tid; i < n_durs; i += nth) {
        const double q = durs[i];
        const bool ok = isfinite(q) && q > 0.0 && q <= 0.5;
        bd += ok ? 0 : 1;
        if (ok) qmax = fmax(qmax, q);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        bp += __shfl_xor_sync(0xffffffffu, bp, o);
        bd += __shfl_xor_sync(0xffffffffu, bd, o);
        qmax = fmax(qmax, __shfl_xor_sync(0xffffffffu, qmax, o));
    }
    if ((threadIdx.x & 31) == 0) {
        if (bp) atomicAdd(&info->bad_period, bp);
        if (bd) atomicAdd(&info->bad_duration, bd);
        // positive doubles order like their bit patterns
        atomicMax((unsigned long long*)&info->q_max, (unsigned long long)__double_as_longlong(qmax));
    }
}

// sum g_D and sum g_D^2 depend on D alone: one warp per D = 1 .. gtab_max, once per search
// (lane-strided sums + shuffle tree: the order every later use relies on).
__global__ void __launch_bounds__(256) k_gtab(const double* __restrict__ tmpl, int n_tmpl, int gtab_max,
                                              double* __restrict__ gtab) {
    const int D = ((blockIdx.x * blockDim.x + threadIdx.x) >> 5) + 1;
    const int lane = threadIdx.x & 31;
    if (D > gtab_max) return;
    double sg = 0.0, sg2 = 0.0;
    for (int j = lane; j < D; j += 32) {
        const double g = tmpl_at(tmpl, n_tmpl, j, D);
        sg += g; sg2 += g * g;
    }
    sg = warp_sum(sg); sg2 = warp_sum(sg2);
    if (lane == 0) { gtab[2 * D] = sg; gtab[2 * D + 1] = sg2; }
}

// One thread per (period, duration): D, stride, mean(g_D), sum g_D^2 (table look-up), duplicate-D flag.
__global__ void __launch_bounds__(256) k_durtab(TileArgs a) {
    const int tr = blockIdx.x * blockDim.x + threadIdx.x;
    if (tr >= a.tile * a.n_dur) return;
    const int pl = tr / a.n_dur, jd = tr % a.n_dur;
    const double* qrow = a.dur_per_period ? a.durs + (a.p0 + pl) * (long long)a.n_dur : a.durs;
    const int D = points_in_duration(qrow[jd], a.n);
    int skip = 0, dmax = D;
    for (int k = 0; k < jd; ++k) {
        const int Dk = points_in_duration(qrow[k], a.n);
        skip |= (Dk == D);
        dmax = max(dmax, Dk);
    }
    if (jd == a.n_dur - 1 && a.x1) {
        // zero margin behind the period's wrap pad (written later by the sort stage, up to n + dmax): the
        // ring kernels copy whole 32-double row windows, which may reach kXMargin entries past the pad
        double* m1 = a.x1 + (long long)pl * a.pitch + a.n + dmax;
        for (int i = 0; i < kXMargin; ++i) m1[i] = 0.0;
        if (!a.uniform) { double* m0 = a.x0 + (long long)pl * a.pitch + a.n + dmax; for (int i = 0; i < kXMargin; ++i) m0[i] = 0.0; }
    }
    double sg = 0.0, sg2 = 0.0;
    if (!skip) {
        if (D <= a.gtab_max) { sg = a.gtab[2 * D]; sg2 = a.gtab[2 * D + 1]; }
        else {                       // beyond the table (not reached: it covers q_max): the same sums, serially
            double p[32], p2[32];
            for (int l = 0; l < 32; ++l) {
                p[l] = 0.0; p2[l] = 0.0;
                for (int j = l; j < D; j += 32) { const double g = tmpl_at(a.tmpl, a.n_tmpl, j, D); p[l] += g; p2[l] += g * g; }
            }
            for (int o = 16; o > 0; o >>= 1)             // the butterfly of warp_sum, lane by lane
                for (int l = 0; l < o; ++l) { p[l] += p[l ^ o]; p2[l] += p2[l ^ o]; }
            sg = p[0]; sg2 = p2[0];
        }
    }
    DurEntry e;
    e.D = D; e.stride = t0_stride(D, a.dt0);
    e.gbar = __ddiv_rn(sg, (double)D); e.gg2 = sg2; e.skip = skip; e.pad_ = 0;
    a.durtab[tr] = e;
}

// chi2 variant of one trial (see chi2_ring.cu): classes of at most 21 taps, ring size, narrow/wide.
__device__ __forceinline__ int chi2_variant(const DurEntry& e, const TileArgs& a) {
    if (e.skip) return -1;
    const int M = (e.D + e.stride - 1) / e.stride;
    const int ncls = chi2_classes(M, e.stride, a.uniform != 0);
    const int stp = ncls * e.stride;
    const int taps = (e.D + stp - 1) / stp;
    const int mbi = chi2_ring_index(taps);
    // narrow path: class stride <= 16; when dy is not uniform its two-ring march takes at most 16 taps
    const int narrow = (stp <= kChi2NarrowMax && (a.uniform || taps <= 16)) ? 1 : 0;
    return narrow * kChi2Rings + mbi;
}

// Trials are binned in order (the trials of a period stay neighbours and share its x1 in L2):
// kBinBlocks CTAs own contiguous segments of the trial range and, inside a CTA, every thread a
// contiguous chunk.  PHASE 0 counts per (CTA, variant) into a.trial_count[kChi2Variants * (1 + b)];
// PHASE 1 adds the counts of the CTAs before it, writes the lists and (last CTA) the totals.
template <int PHASE>
__global__ void __launch_bounds__(256) k_bin_trials(TileArgs a) {
    __shared__ int s_warp[kChi2Variants][8];
    __shared__ int s_base[kChi2Variants];
    const int T = a.tile * a.n_dur;
    const int seg = (T + gridDim.x - 1) / gridDim.x;
    const int b0 = min(T, (int)blockIdx.x * seg), b1 = min(T, b0 + seg);
    const int chunk = (b1 - b0 + blockDim.x - 1) / blockDim.x;
    const int t0 = min(b1, b0 + (int)threadIdx.x * chunk), t1 = min(b1, t0 + chunk);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int* block_counts = a.trial_count + kChi2Variants;
    int cnt[kChi2Variants];
#pragma unroll
    for (int v = 0; v < kChi2Variants; ++v) cnt[v] = 0;
    for (int t = t0; t < t1; ++t) {
        const int v = chi2_variant(a.durtab[t], a);
#pragma unroll
        for (int k = 0; k < kChi2Variants; ++k) cnt[k] += (v == k) ? 1 : 0;
        if (PHASE == 0 && v < 0) { Partial p; p.dchi2 = 0.0; p.depth = 0.0; p.start = 0; p.valid = 0; a.partial[t] = p; }
    }
    if (PHASE == 1 && threadIdx.x < kChi2Variants) {
        int base = 0;
        for (int b = 0; b < (int)blockIdx.x; ++b) base += block_counts[b * kChi2Variants + threadIdx.x];
        s_base[threadIdx.x] = base;
    }
    int excl[kChi2Variants];
#pragma unroll
    for (int v = 0; v < kChi2Variants; ++v) {
        int x = cnt[v];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
        excl[v] = x - cnt[v];
        if (lane == 31) s_warp[v][warp] = x;
    }
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int v = 0; v < kChi2Variants; ++v) {
            const int c = lane < (int)(blockDim.x >> 5) ? s_warp[v][lane & 7] : 0;
            int x = c;
#pragma unroll
            for (int o = 1; o < 8; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
            if (lane < 8) s_warp[v][lane] = x - c;
            if (lane == 7) {
                if (PHASE == 0) block_counts[blockIdx.x * kChi2Variants + v] = x;
                else if (blockIdx.x == gridDim.x - 1) {
                    a.trial_count[v] = s_base[v] + x;
                    a.trial_count[kChi2Variants * (1 + kBinBlocks) + v] = 0;     // the variant's trial queue (chi2_ring.cu)
                }
            }
        }
    }
    if (PHASE == 0) return;
    __syncthreads();
    int pos[kChi2Variants];
#pragma unroll
    for (int v = 0; v < kChi2Variants; ++v) pos[v] = s_base[v] + s_warp[v][warp] + excl[v];
    for (int t = t0; t < t1; ++t) {
        const int v = chi2_variant(a.durtab[t], a);
#pragma unroll
        for (int k = 0; k < kChi2Variants; ++k)
            if (v == k) { a.trial_list[(long long)k * T + pos[k]] = t; ++pos[k]; }
    }
}

}  // namespace

// survey mode: blockIdx.y = curve; periods [per_off[c], per_off[c+1]) and, when dur_per_period, their rows
__global__ void __launch_bounds__(256) k_grid_check_batch(const double* __restrict__ periods,
                                                          const long long* __restrict__ per_off,
                                                          const double* __restrict__ durs, int n_dur,
                                                          int dur_per_period, CurveInfo* info) {
    const int c = blockIdx.y;
    const long long p0 = per_off[c], np = per_off[c + 1] - p0;
    int bp = 0, bd = 0;
    double qmax = 0.0;
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long nth = (long long)gridDim.x * blockDim.x;
    for (long long i = tid; i < np; i += nth) {
        const double p = periods[p0 + i];
        bp += (isfinite(p) && p > 0.0) ? 0 : 1;
    }
    const long long nd = dur_per_period ? np * n_dur : n_dur;
    const double* dq = dur_per_period ? durs + p0 * n_dur : durs;
    for (long long i = tid; i < nd; i += nth) {
        const double q = dq[i];
        const bool ok = isfinite(q) && q > 0.0 && q <= 0.5;
        bd += ok ? 0 : 1;
        if (ok) qmax = fmax(qmax, q);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        bp += __shfl_xor_sync(0xffffffffu, bp, o);
        bd += __shfl_xor_sync(0xffffffffu, bd, o);
        qmax = fmax(qmax, __shfl_xor_sync(0xffffffffu, qmax, o));
    }
    if ((threadIdx.x & 31) == 0) {
        if (bp) atomicAdd(&info[c].bad_period, bp);
        if (bd) atomicAdd(&info[c].bad_duration, bd);
        atomicMax((unsigned long long*)&info[c].q_max, (unsigned long long)__double_as_longlong(qmax));
    }
}

void launch_curve_pre(const double* t, const double* y, const double* dy, int n, double* wr,
                      double* w, double* wr2, CurveInfo* info, cudaStream_t st) {
    k_curve_pre<<<1, 1024, 0, st>>>(t, y, dy, n, wr, w, wr2, info);
}

void launch_grid_check(const double* periods, long long n_per, const double* durs,
                       long long n_durs_total, CurveInfo* info, cudaStream_t st) {
    long long work = n_durs_total > n_per ? n_durs_total : n_per;
    int blocks = (int)((work + 256 * 8 - 1) / (256 * 8));
    blocks = blocks < 1 ? 1 : (blocks > 1184 ? 1184 : blocks);
    k_grid_check<<<blocks, 256, 0, st>>>(periods, n_per, durs, n_durs_total, info);
}

void launch_batch_pre(int n_curves, const double* t, const double* y, const double* dy, const long long* curve_off,
                      const double* periods, const long long* per_off, const double* durs, int n_dur,
                      int dur_per_period, double* wr, double* w, double* wr2, CurveInfo* info, cudaStream_t st) {
    k_curve_pre_batch<<<n_curves, 1024, 0, st>>>(t, y, dy, curve_off, wr, w, wr2, info);
    k_grid_check_batch<<<dim3(8, n_curves), 256, 0, st>>>(periods, per_off, durs, n_dur, dur_per_period, info);
}

void launch_bin_trials(const TileArgs& a, cudaStream_t st) {
    k_bin_trials<0><<<kBinBlocks, 256, 0, st>>>(a);
    k_bin_trials<1><<<kBinBlocks, 256, 0, st>>>(a);
}

void launch_gtab(const double* tmpl, int n_tmpl, int gtab_max, double* gtab, cudaStream_t st) {
    const int blocks = (int)(((long long)gtab_max * 32 + 255) / 256);
    k_gtab<<<blocks, 256, 0, st>>>(tmpl, n_tmpl, gtab_max, gtab);
}

void launch_durtab(const TileArgs& a, cudaStream_t st) {
    const long long trials = (long long)a.tile * a.n_dur;
    k_durtab<<<(int)((trials + 255) / 256), 256, 0, st>>>(a);
}

}  // namespace gtls
