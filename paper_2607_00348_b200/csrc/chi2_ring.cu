// Steps a5-a8, in-transit chi2 as a register-ring correlation -- the dominant kernel.
//
// For one (period, duration) with D points per window and stride st between trial starts
// (Eq. 18), split the template index j = m*st + i (tap m < M = ceil(D/st),
// column i < st).  With the folded curve viewed as rows of st points, X[rho][i] = x1[rho*st+i],
//     C[k] = sum_i sum_m g[m*st+i] * X[k+m][i]                              (Eq. 16)
// is, per column i, a 1-D correlation along the rows with the M taps g[m*st+i].
//
// A lane owns ONE column and marches down its rows holding MB taps and a ring of MB window
// accumulators in registers: every X value is loaded from L2 exactly once (coalesced across the
// lanes of a warp, software-prefetched one block of MB rows ahead) and feeds MB DFMAs; each row
// step starts one window (DMUL) and completes one.  There is no shared-memory staging of X and no
// CTA barrier in the hot loop -- the FP64 pipe (64 DFMA/clk/SM) is the only busy resource:
// 1 LDG.64 + 1 STS.64 per MB DFMAs.  Completed per-column sums go through a small per-warp
// shared-memory buffer once per MB rows, are summed over the columns of a window in fixed order
// (deterministic) and land in a per-CTA table Cpart; M > MB is handled by looping tap blocks.
//
// Lanes are assigned from a flat list of (row segment, column) pairs, so warps are full for
// every st (32 consecutive entries span at most ceil(31/st)+1 segments).  The segment count is
// chosen per trial to balance the 4 warps of the CTA against the MB-1 halo rows each segment
// needs before its first window completes.
//
// a5 (depth from the prefix sums, Eq. 12-14), the score dchi2 = -2 a C + a^2 G (a6+a7; the
// S2 window term of Eq. 15 cancels against the same term of Eq. 16) and the lexicographic
// (dchi2, start) argmin (a8) run per window tile from Cpart.
// The template nodes are staged in shared memory with one TMA bulk copy (cp.async.bulk).
#include "gtls_internal.cuh"

namespace gtls {

namespace {

constexpr int kRT = 128;                 // threads per CTA
constexpr int kRW = kRT / 32;            // warps per CTA
constexpr int kPartPitch = 33;           // doubles per slot row of the per-warp emit buffer
constexpr int kMBMax = 21;
constexpr int kCDoubles = 5120;          // Cpart capacity (40 KB)
constexpr int kTmplSmem = 1024;          // template nodes cached in shared memory
constexpr int kMaxSeg = 512;

struct Cand { double d; double depth; int s; int has; };

__device__ __forceinline__ void cand_offer(Cand& b, double d, int s, double depth) {
    if (!b.has || d < b.d || (d == b.d && s < b.s)) { b.d = d; b.s = s; b.depth = depth; b.has = 1; }
}

struct RGeom {
    int D, st, nW, M, MB, nmb, J, Kt;
    double tscale;                       // (n_tmpl - 1) / D
};

// tap-block size for M taps: the instantiated MB that wastes the fewest padded taps
__device__ __forceinline__ void pick_mb(int M, int& MB, int& nmb) {
    const int cand[5] = {21, 16, 12, 8, 4};
    int best = 1 << 30;
    MB = 21; nmb = 1;
#pragma unroll
    for (int c = 0; c < 5; ++c) {
        const int nb = (M + cand[c] - 1) / cand[c];
        const int cost = nb * cand[c] + (nb - 1);        // slight preference for fewer blocks
        if (cost < best) { best = cost; MB = cand[c]; nmb = nb; }
    }
}

struct Item {                            // one warp work item: 32 flat (segment, column) slots
    int f0;                              // first flat slot
    int seg_first, ng;                   // segments touched by this warp
    int idx;                             // item index (= f0 / 32)
};

// One tap block of one item: march `nblk` blocks of MB rows.  `xp` points at this lane's X value of
// the first row, rows >= rows_valid read as 0.  After each block the MB completed window sums of
// every lane sit in `part` (slot-major); the warp reduces them over the lanes of each segment and
// stores / accumulates into cpart[j * Kt + window].
template <int MB>
__device__ __forceinline__ void march(const double* __restrict__ xp, const int st, const int rows_valid,
                                      const int nblk, const double (&T)[MB], double* __restrict__ part,
                                      const int lane, const Item it, const int slots, const int L,
                                      const int nWt, const int Kt, double* __restrict__ cpart,
                                      const bool first) {
    double acc[MB], xc[MB], xn[MB];
#pragma unroll
    for (int u = 0; u < MB; ++u) {
        acc[u] = 0.0;
        xn[u] = u < rows_valid ? __ldg(xp) : 0.0;
        xp += st;
    }
    double* const pl = part + lane;
    for (int blk = 0; blk < nblk; ++blk) {
        const int gnext = (blk + 1) * MB;
#pragma unroll
        for (int u = 0; u < MB; ++u) {
            xc[u] = xn[u];
            xn[u] = (blk + 1 < nblk && gnext + u < rows_valid) ? __ldg(xp) : 0.0;   // next block, in flight
            xp += st;
        }
#pragma unroll
        for (int u = 0; u < MB; ++u) {
#pragma unroll
            for (int m = 0; m < MB; ++m) {
                const int a = (u - m + MB) % MB;
                if (m == 0) acc[a] = T[0] * xc[u];                  // window gamma starts at this row
                else acc[a] = fma(T[m], xc[u], acc[a]);
            }
            pl[u * kPartPitch] = acc[(u + 1) % MB];                 // window gamma - (MB-1) is complete
        }
        __syncwarp();
        for (int t = lane; t < it.ng * MB; t += 32) {
            const int gi = t / MB, slot = t - gi * MB;
            const int seg = it.seg_first + gi;
            const int kw = blk * MB + slot - (MB - 1);
            const int w = seg * L + kw;
            if (kw >= 0 && kw < L && w < nWt) {
                int lo = seg * st - it.f0, hi = lo + st;
                lo = lo < 0 ? 0 : lo;
                hi = hi > 32 ? 32 : hi;
                hi = hi > slots - it.f0 ? slots - it.f0 : hi;
                const double* pr = part + slot * kPartPitch;
                double s0 = 0.0, s1 = 0.0;
                int q = lo;
                for (; q + 1 < hi; q += 2) { s0 += pr[q]; s1 += pr[q + 1]; }
                if (q < hi) s0 += pr[q];
                const double sum = s0 + s1;
                const int j = it.idx - ((seg * st) >> 5);
                double* dst = cpart + j * Kt + w;
                *dst = first ? sum : *dst + sum;
            }
        }
        __syncwarp();
    }
}

__device__ __forceinline__ double tmpl_lerp(const double* __restrict__ tm, int n_tmpl, int j, double tscale) {
    const double u = ((double)j + 0.5) * tscale;
    int k = (int)u;                                   // u >= 0: truncation == floor
    k = k > n_tmpl - 2 ? n_tmpl - 2 : k;
    const double fr = u - (double)k;
    const double t0 = tm[k];
    return t0 + fr * (tm[k + 1] - t0);
}

template <int MB>
__device__ __forceinline__ void run_item(const TileArgs& a, const RGeom& q, const double* __restrict__ tm,
                                         const double* __restrict__ x, const bool square,
                                         const Item it, const int lane, const int slots, const int L,
                                         const int nWt, const int k0, double* __restrict__ part,
                                         double* __restrict__ cpart) {
    const int f = it.f0 + lane;
    const bool active = f < slots;
    const int seg = active ? f / q.st : 0;
    const int col = active ? f - seg * q.st : 0;
    const int nblk = (L + MB - 1 + MB - 1) / MB;
    const long long lim = (long long)a.n + q.D;       // x entries >= lim are never needed
    for (int b = 0; b < q.nmb; ++b) {
        double T[MB];
#pragma unroll
        for (int m = 0; m < MB; ++m) {
            const long long j = (long long)(b * MB + m) * q.st + col;
            double g = 0.0;
            if (active && j < q.D) g = tmpl_lerp(tm, a.n_tmpl, (int)j, q.tscale);
            T[m] = square ? g * g : g;
        }
        const long long ebase = ((long long)(k0 + seg * L) + (long long)b * MB) * q.st + col;
        int rows_valid = 0;
        if (active && ebase < lim) {
            const long long rv = (lim - ebase + q.st - 1) / q.st;
            rows_valid = rv > (long long)nblk * MB ? nblk * MB : (int)rv;
        }
        march<MB>(x + (active ? ebase : 0), q.st, rows_valid, nblk, T, part, lane, it, slots, L, nWt,
                  q.Kt, cpart, b == 0);
    }
}

template <bool UNIFORM>
__global__ void __launch_bounds__(kRT) k_chi2_ring(TileArgs a) {
    extern __shared__ double dsm[];                 // [kRW][kMBMax*kPartPitch] emit buffers, then Cpart
    __shared__ __align__(16) double s_tmpl[kTmplSmem];
    double* const s_cpart = dsm + kRW * kMBMax * kPartPitch;
    __shared__ RGeom s_q;
    __shared__ Cand s_best[kRW];
    __shared__ int s_cost[kRW], s_nseg[kRW];
    __shared__ __align__(8) unsigned long long s_mbar;

    const int jd = blockIdx.x, pl = blockIdx.y;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const DurEntry e = a.durtab[(long long)pl * a.n_dur + jd];
    Partial* out = a.partial + (long long)pl * a.n_dur + jd;
    if (e.skip) {
        if (tid == 0) { out->valid = 0; out->dchi2 = 0.0; out->depth = 0.0; out->start = 0; }
        return;
    }
    // ---- template nodes -> shared memory: one TMA bulk copy when size / alignment allow ------
    const bool tmpl_in_smem = a.n_tmpl <= kTmplSmem;
    const unsigned tbytes = (unsigned)a.n_tmpl * 8u;
    const bool tma_ok = tmpl_in_smem && (tbytes % 16u == 0) && (((unsigned long long)a.tmpl & 15ull) == 0);
    if (tma_ok) {
        const unsigned mb = (unsigned)__cvta_generic_to_shared(&s_mbar);
        if (tid == 0) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mb));
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mb), "r"(tbytes) : "memory");
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"((unsigned)__cvta_generic_to_shared(s_tmpl)), "l"(a.tmpl), "r"(tbytes), "r"(mb)
                         : "memory");
        }
    } else if (tmpl_in_smem) {
        for (int k = tid; k < a.n_tmpl; k += kRT) s_tmpl[k] = a.tmpl[k];
    }
    if (tid == 0) {
        RGeom q;
        q.D = e.D; q.st = e.stride;
        q.nW = (a.n + q.st - 1) / q.st;
        q.M = (q.D + q.st - 1) / q.st;
        pick_mb(q.M, q.MB, q.nmb);
        q.J = (q.st + 30) / 32 + 1;                    // warps that can cover one segment's st slots
        q.Kt = kCDoubles / (q.J * (UNIFORM ? 1 : 2));
        q.tscale = __ddiv_rn((double)(a.n_tmpl - 1), (double)q.D);
        s_q = q;
    }
    __syncthreads();
    if (tma_ok) {
        const unsigned mb = (unsigned)__cvta_generic_to_shared(&s_mbar);
        unsigned done = 0;
        while (!done) {
            asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\nselp.u32 %0, 1, 0, p;\n}"
                         : "=r"(done) : "r"(mb) : "memory");
        }
    }
    const RGeom q = s_q;
    const double* __restrict__ tm = tmpl_in_smem ? s_tmpl : a.tmpl;
    const double* __restrict__ x1 = a.x1 + (long long)pl * a.pitch;
    const double* __restrict__ x0 = a.x0 + (long long)pl * a.pitch;
    const double* __restrict__ s1 = a.s1 + (long long)pl * a.spitch;
    const double* __restrict__ s0 = a.s0 + (long long)pl * a.spitch;
    const double G_u = a.w_uniform * e.gg2, sw_u = (double)q.D * a.w_uniform;
    double* part = dsm + warp * (kMBMax * kPartPitch);
    Cand best; best.has = 0; best.d = 0.0; best.s = 0; best.depth = 0.0;

    for (int k0 = 0; k0 < q.nW; k0 += q.Kt) {
        const int nWt = min(q.Kt, q.nW - k0);
        // ---- segment count: minimise rounds(items / warps) * rows per item ----------------------
        int bc = 0x7fffffff, bn = 1;
        for (int ns = tid + 1; ns <= kMaxSeg && ns <= nWt; ns += kRT) {
            const int L = (nWt + ns - 1) / ns;
            const int items = (ns * q.st + 31) >> 5;
            const int rounds = (items + kRW - 1) / kRW;
            const int cost = rounds * (((L + 2 * q.MB - 2) / q.MB) * q.MB + 6);
            if (cost < bc) { bc = cost; bn = ns; }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const int oc = __shfl_xor_sync(0xffffffffu, bc, o), on = __shfl_xor_sync(0xffffffffu, bn, o);
            if (oc < bc || (oc == bc && on < bn)) { bc = oc; bn = on; }
        }
        if (lane == 0) { s_cost[warp] = bc; s_nseg[warp] = bn; }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < kRW; ++k)
            if (s_cost[k] < bc || (s_cost[k] == bc && s_nseg[k] < bn)) { bc = s_cost[k]; bn = s_nseg[k]; }
        const int nseg = bn;
        const int L = (nWt + nseg - 1) / nseg;
        const int slots = nseg * q.st;
        const int items = (slots + 31) >> 5;

        for (int pass = 0; pass < (UNIFORM ? 1 : 2); ++pass) {
            const double* __restrict__ x = pass == 0 ? x1 : x0;
            double* cpart = s_cpart + pass * q.J * q.Kt;
            for (int i = warp; i < items; i += kRW) {
                Item it;
                it.idx = i; it.f0 = i << 5;
                it.seg_first = it.f0 / q.st;
                const int last = min(it.f0 + 31, slots - 1) / q.st;
                it.ng = last - it.seg_first + 1;
                switch (q.MB) {
                    case 21: run_item<21>(a, q, tm, x, pass == 1, it, lane, slots, L, nWt, k0, part, cpart); break;
                    case 16: run_item<16>(a, q, tm, x, pass == 1, it, lane, slots, L, nWt, k0, part, cpart); break;
                    case 12: run_item<12>(a, q, tm, x, pass == 1, it, lane, slots, L, nWt, k0, part, cpart); break;
                    case 8: run_item<8>(a, q, tm, x, pass == 1, it, lane, slots, L, nWt, k0, part, cpart); break;
                    default: run_item<4>(a, q, tm, x, pass == 1, it, lane, slots, L, nWt, k0, part, cpart); break;
                }
            }
        }
        __syncthreads();
        // ---- a5 + a8 per window of the tile ---------------------------------------------------------
        for (int w = tid; w < nWt; w += kRT) {
            const int seg = w / L;
            const int fw = (seg * q.st) >> 5, lw = (seg * q.st + q.st - 1) >> 5;
            double C = 0.0, Gs = 0.0;
            for (int j = 0; j <= lw - fw; ++j) {
                C += s_cpart[j * q.Kt + w];
                if (!UNIFORM) Gs += s_cpart[(q.J + j) * q.Kt + w];
            }
            const int sidx = (k0 + w) * q.st;
            const double swr = s1[sidx + q.D] - s1[sidx];
            const double sw = UNIFORM ? sw_u : s0[sidx + q.D] - s0[sidx];
            const double rbar = __ddiv_rn(swr, sw);
            const double depth = __ddiv_rn(fmax(rbar, 0.0), e.gbar);
            const double Gv = UNIFORM ? G_u : Gs;
            const double d = -2.0 * depth * C + (depth * depth) * Gv;
            cand_offer(best, d, sidx, depth);
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
    if (tid == 0) {
        for (int k = 1; k < kRW; ++k)
            if (s_best[k].has) cand_offer(best, s_best[k].d, s_best[k].s, s_best[k].depth);
        out->valid = best.has; out->dchi2 = best.d; out->depth = best.depth; out->start = best.s;
    }
}

}  // namespace

void launch_chi2_ring(const TileArgs& a, cudaStream_t st) {
    const dim3 grid(a.n_dur, a.tile);
    const size_t sm = (size_t)(kRW * kMBMax * kPartPitch + kCDoubles) * sizeof(double);
    static bool set = false;
    if (!set) {
        cudaFuncSetAttribute(k_chi2_ring<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
        cudaFuncSetAttribute(k_chi2_ring<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
        set = true;
    }
    if (a.uniform) k_chi2_ring<true><<<grid, kRT, sm, st>>>(a);
    else k_chi2_ring<false><<<grid, kRT, sm, st>>>(a);
}

}  // namespace gtls
