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

constexpr int kPartPitch = 33;           // doubles per slot row of the per-warp emit buffer
constexpr int kMBMax = 21;

// rows prefetched ahead of the FMAs (divides MB)
template <int MB> struct PfRows { static constexpr int v = (MB % 7 == 0) ? 7 : (MB >= 8 ? MB / 2 : MB); };

__device__ __forceinline__ double lds64(const unsigned addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts64(const unsigned addr, const double v) {
    asm volatile("st.shared.f64 [%0], %1;" ::"r"(addr), "d"(v) : "memory");
}

struct EmitCtx {                         // where completed window sums of one item go
    int idx, f0, seg_first, ng;          // item index, first flat slot, segments touched by the warp
    int slots, st, L, nWt, Kt;
    bool first;                          // first tap block: store, else accumulate
    double* cpart;
    unsigned part;                       // shared-space address of the per-warp [MB][kPartPitch] buffer
};

__device__ __forceinline__ void cpart_put(const EmitCtx& c, const int seg, const int kw, const double sum) {
    const int w = seg * c.L + kw;
    if (kw >= 0 && kw < c.L && w < c.nWt) {
        const int j = c.idx - ((seg * c.st) >> 5);
        double* dst = c.cpart + j * c.Kt + w;
        *dst = c.first ? sum : *dst + sum;
    }
}

// The MB completed window sums of every lane sit in part[slot][lane]; sum them over the lanes of
// each segment in fixed order.  One segment per warp (the common case): lane = slot, 32 loads in
// four independent chains.  Otherwise: one (segment, slot) task per lane and round.
template <int MB>
__device__ __forceinline__ void reduce_block(const EmitCtx& c, const int kw0, const int lane) {
    __syncwarp();
    if (c.ng == 1) {
        if (lane < MB) {
            const unsigned pr = c.part + (unsigned)(lane * kPartPitch * 8);
            double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
#pragma unroll
            for (int q = 0; q < 32; q += 4) {
                s0 += lds64(pr + 8 * q);
                s1 += lds64(pr + 8 * q + 8);
                s2 += lds64(pr + 8 * q + 16);
                s3 += lds64(pr + 8 * q + 24);
            }
            cpart_put(c, c.seg_first, kw0 + lane, (s0 + s1) + (s2 + s3));
        }
    } else {
        for (int t = lane; t < c.ng * MB; t += 32) {
            const int gi = t / MB, sl = t - gi * MB;
            const int seg = c.seg_first + gi;
            int lo = seg * c.st - c.f0, hi = lo + c.st;
            lo = lo < 0 ? 0 : lo;
            hi = hi > 32 ? 32 : hi;
            hi = hi > c.slots - c.f0 ? c.slots - c.f0 : hi;
            const unsigned pr = c.part + (unsigned)(sl * kPartPitch * 8);
            double s0 = 0.0, s1 = 0.0;
            int q = lo;
            for (; q + 1 < hi; q += 2) { s0 += lds64(pr + 8 * q); s1 += lds64(pr + 8 * q + 8); }
            if (q < hi) s0 += lds64(pr + 8 * q);
            cpart_put(c, seg, kw0 + sl, s0 + s1);
        }
    }
    __syncwarp();
}

// One tap block of one item: march `nblk` blocks of MB rows.  `xp` points at this lane's X value of
// the first row; rows >= rows_valid read as 0.  PF rows are in flight ahead of the FMAs; after every
// block of MB rows the MB completed window sums are reduced over the lanes of each segment.
template <int MB>
__device__ __forceinline__ void march(const double* __restrict__ xp, const int st, const int rows_valid,
                                      const int nblk, const double (&T)[MB], const int lane,
                                      const EmitCtx& c) {
    constexpr int PF = PfRows<MB>::v;
    double acc[MB], xr[PF];
#pragma unroll
    for (int u = 0; u < MB; ++u) acc[u] = 0.0;
#pragma unroll
    for (int u = 0; u < PF; ++u) {
        xr[u] = u < rows_valid ? __ldg(xp) : 0.0;
        xp += st;
    }
    int row_pf = PF;                               // row index the next prefetch belongs to
    const unsigned pl = c.part + (unsigned)(lane * 8);
#pragma unroll 1
    for (int blk = 0; blk < nblk; ++blk) {
#pragma unroll
        for (int u = 0; u < MB; ++u) {
            const double x = xr[u % PF];
            xr[u % PF] = row_pf < rows_valid ? __ldg(xp) : 0.0;
            xp += st;
            ++row_pf;
#pragma unroll
            for (int m = 0; m < MB; ++m) {
                const int a = (u - m + MB) % MB;
                if (m == 0) acc[a] = T[0] * x;                      // window gamma starts at this row
                else acc[a] = fma(T[m], x, acc[a]);
            }
            sts64(pl + (unsigned)(u * kPartPitch * 8), acc[(u + 1) % MB]);   // window gamma-(MB-1) complete
        }
        reduce_block<MB>(c, blk * MB - (MB - 1), lane);
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
                                         const double* __restrict__ x, const bool square, const int item,
                                         const int lane, const int slots, const int L, const int nWt,
                                         const int k0, const unsigned part, double* __restrict__ cpart) {
    EmitCtx c;
    c.idx = item; c.f0 = item << 5;
    c.seg_first = c.f0 / q.st;
    c.ng = min(c.f0 + 31, slots - 1) / q.st - c.seg_first + 1;
    c.slots = slots; c.st = q.st; c.L = L; c.nWt = nWt; c.Kt = q.Kt;
    c.cpart = cpart; c.part = part;
    const int f = c.f0 + lane;
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
        c.first = b == 0;
        march<MB>(x + (active ? ebase : 0), q.st, rows_valid, nblk, T, lane, c);
    }
}

template <bool UNIFORM>
__global__ void __launch_bounds__(kRT, 3) k_chi2_ring(TileArgs a) {
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
    const unsigned part = (unsigned)__cvta_generic_to_shared(dsm + warp * (kMBMax * kPartPitch));
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
                switch (q.MB) {
                    case 21: run_item<21>(a, q, tm, x, pass == 1, i, lane, slots, L, nWt, k0, part, cpart); break;
                    case 16: run_item<16>(a, q, tm, x, pass == 1, i, lane, slots, L, nWt, k0, part, cpart); break;
                    case 12: run_item<12>(a, q, tm, x, pass == 1, i, lane, slots, L, nWt, k0, part, cpart); break;
                    case 8: run_item<8>(a, q, tm, x, pass == 1, i, lane, slots, L, nWt, k0, part, cpart); break;
                    default: run_item<4>(a, q, tm, x, pass == 1, i, lane, slots, L, nWt, k0, part, cpart); break;
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
