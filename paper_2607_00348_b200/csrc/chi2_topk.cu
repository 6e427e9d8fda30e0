// Pruning variant of steps a5-a8 (reading G19, gtls_opts.top_k = K > 0): for every (period, duration)
// the running mean rbar = sum_W w r / sum_W w (Eq. 12-14) is taken at ALL strided
// starts from the prefix sums, the K deepest starts are kept (ties -> lower start) and chi2 is
// evaluated only there, by direct sums of the template over the window (Eq. 16).
// north_star words the search this way ("running mean ... to find the deepest positions"); the paper
// itself evaluates every trial position, which is the default path (chi2_ring.cu).
//
// One warp per trial.  Pass 1: every lane scans its share of the starts and keeps its K deepest in
// registers (insertion into a sorted list; a later equal value does not displace an earlier one).
// Pass 2: K rounds of a warp-wide argmax over the lanes' list heads (value descending, start
// ascending); the winner's window is evaluated at once by the whole warp: C = sum_j g_D[j] x1[s+j]
// (lane-strided partial sums, shuffle tree: deterministic), G likewise or w * sum g_D^2 when dy is
// uniform, dchi2 = -2 a C + a^2 G with a = max(rbar, 0) / mean(g_D).
#include "gtls_internal.cuh"

namespace gtls {

namespace {

__device__ __forceinline__ double warp_sum_d(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__global__ void __launch_bounds__(128) k_chi2_topk(TileArgs a) {
    const int trial = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (trial >= a.tile * a.n_dur) return;
    const DurEntry e = a.durtab[trial];
    Partial* out = a.partial + trial;
    if (e.skip) {                                   // same D as an earlier duration of this period
        if (lane == 0) { out->valid = 0; out->dchi2 = 0.0; out->depth = 0.0; out->start = 0; }
        return;
    }
    const int pl = trial / a.n_dur;
    const double* __restrict__ s1 = a.s1 + (long long)pl * a.spitch;
    const double* __restrict__ s0 = a.s0 + (long long)pl * a.spitch;
    const double* __restrict__ x1 = a.x1 + (long long)pl * a.pitch;
    const double* __restrict__ x0 = a.x0 + (long long)pl * a.pitch;
    const int D = e.D, st = e.stride;
    const int nW = (a.n + st - 1) / st;
    const int K = a.top_k < kTopKMax ? a.top_k : kTopKMax;
    const double sw_u = (double)D * a.w_uniform;
    const double ninf = __longlong_as_double((long long)0xfff0000000000000ULL);

    // ---- pass 1: the lane's K deepest starts, sorted (value descending, start ascending) --------
    double tv[kTopKMax];
    int tk[kTopKMax];
#pragma unroll
    for (int i = 0; i < kTopKMax; ++i) { tv[i] = ninf; tk[i] = 0x7fffffff; }
    for (int k = lane; k < nW; k += 32) {
        const int s = k * st;
        const double swr = s1[s + D] - s1[s];
        const double sw = a.uniform ? sw_u : s0[s + D] - s0[s];
        double v = __ddiv_rn(swr, sw);
        int vk = k;
        // insertion: v goes in front of the first entry that is smaller (an earlier start wins a tie);
        // from there on every entry moves down one place
        bool moving = false;
#pragma unroll
        for (int i = 0; i < kTopKMax; ++i) {
            if (i < K && (moving || v > tv[i])) {
                moving = true;
                const double tvv = tv[i]; const int tkk = tk[i];
                tv[i] = v; tk[i] = vk;
                v = tvv; vk = tkk;
            }
        }
    }

    // ---- pass 2: K rounds of warp argmax over the list heads, each winner evaluated at once ------
    const int rounds = K < nW ? K : nW;
    double bd = 0.0, bdepth = 0.0;
    int bs = 0, has = 0;
    for (int r = 0; r < rounds; ++r) {
        double hv = tv[0];
        int hk = tk[0], hl = lane;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double ov = __shfl_xor_sync(0xffffffffu, hv, o);
            const int ok = __shfl_xor_sync(0xffffffffu, hk, o);
            const int ol = __shfl_xor_sync(0xffffffffu, hl, o);
            if (ov > hv || (ov == hv && ok < hk)) { hv = ov; hk = ok; hl = ol; }
        }
        if (lane == hl) {                           // pop the winner's head
#pragma unroll
            for (int i = 0; i + 1 < kTopKMax; ++i) { tv[i] = tv[i + 1]; tk[i] = tk[i + 1]; }
            tv[kTopKMax - 1] = ninf; tk[kTopKMax - 1] = 0x7fffffff;
        }
        const int s = hk * st;
        const double depth = __ddiv_rn(fmax(hv, 0.0), e.gbar);
        double c = 0.0, g2 = 0.0;
        for (int j = lane; j < D; j += 32) {
            const double g = tmpl_at(a.tmpl, a.n_tmpl, j, D);
            c += g * x1[s + j];
            if (!a.uniform) g2 += (g * g) * x0[s + j];
        }
        c = warp_sum_d(c);
        const double G = a.uniform ? a.w_uniform * e.gg2 : warp_sum_d(g2);
        const double d = -2.0 * depth * c + (depth * depth) * G;
        if (!has || d < bd || (d == bd && s < bs)) { bd = d; bs = s; bdepth = depth; has = 1; }
    }
    if (lane == 0) { out->valid = has; out->dchi2 = bd; out->depth = bdepth; out->start = bs; }
}

}  // namespace

void launch_chi2_topk(const TileArgs& a, cudaStream_t st) {
    const long long warps = (long long)a.tile * a.n_dur;
    k_chi2_topk<<<(int)((warps * 32 + 127) / 128), 128, 0, st>>>(a);
}

}  // namespace gtls
