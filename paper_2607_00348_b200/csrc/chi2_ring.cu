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
// lanes of a warp, software-prefetched a few rows ahead) and feeds MB DFMAs; each row step starts
// one window (DMUL) and completes one.  There is no shared-memory staging of X: the FP64 pipe
// (64 DFMA/clk/SM) is the only busy resource, 1 LDG.64 + 1 STS.64 per MB DFMAs.  After every MB
// rows the MB completed per-column sums of the 32 lanes are summed over the columns of a window in
// fixed order (deterministic) through a per-warp shared-memory buffer and added to the warp's
// window table C[k]; M > MB is handled by looping tap blocks.
//
// ONE WARP OWNS ONE TRIAL (period, duration) from its first row to its argmin: there is no CTA
// barrier after the template nodes are staged, so the warps of an SM (3 CTAs x 4 warps) sit in
// different phases and the scoring epilogue of one hides behind the DFMAs of the others.
// Lanes are assigned from a flat list of (row segment, column) pairs, so warps are full for every
// st; the segment count is chosen per trial to balance lane use against the MB-1 halo rows each
// segment needs before its first window completes.
//
// a5 (depth from the prefix sums, Eq. 12-14), the score dchi2 = -2 a C + a^2 G (a6+a7; the
// S2 window term of Eq. 15 cancels against the same term of Eq. 16) and the lexicographic
// (dchi2, start) argmin (a8) run per window tile from C[k].
// The template nodes are staged in shared memory with one TMA bulk copy (cp.async.bulk).
#include "gtls_internal.cuh"

namespace gtls {

namespace {

constexpr int kRT = 128;                 // threads per CTA
constexpr int kRW = kRT / 32;            // warps (= trials) per CTA
constexpr int kPartPitch = 33;           // doubles per slot row of the per-warp emit buffer
constexpr int kMBMax = 21;
constexpr int kCW = 672;                 // window-table doubles per warp
constexpr int kTmplSmem = 1024;          // template nodes cached in shared memory
constexpr int kFifoBatches = 3;          // batches of PfRows rows per lane in the cp.async FIFO
constexpr int kFifoRows = 24;            // >= kFifoBatches * max PfRows
constexpr int kWarpSmem = kMBMax * kPartPitch + kFifoRows * 32 + kCW;   // doubles of dynamic smem per warp

struct Cand { double d; double depth; int s; int has; };

__device__ __forceinline__ void cand_offer(Cand& b, double d, int s, double depth) {
    if (!b.has || d < b.d || (d == b.d && s < b.s)) { b.d = d; b.s = s; b.depth = depth; b.has = 1; }
}

struct RGeom {
    int D, st, nW, M, MB, nmb, Kt;
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

// 8-byte asynchronous global -> shared copy; `valid == false` writes zeros without reading
__device__ __forceinline__ void cp_async8(const unsigned dst, const double* src, const bool valid) {
    const int sz = valid ? 8 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(dst), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

struct EmitCtx {                         // where completed window sums of one item go
    int f0, seg_first, ng;               // first flat slot, first segment / segments touched by the warp
    int split;                           // ng <= 2: first lane of the second segment (32 if none)
    int slots, st, L, nWt;
    unsigned ctab;                       // shared-space address of the window table (C or G)
    unsigned part;                       // shared-space address of the per-warp [MB][kPartPitch] buffer
    unsigned fifo;                       // shared-space address of the per-warp [kFifoRows][32] X FIFO
};

__device__ __forceinline__ void ctab_add(const EmitCtx& c, const int seg, const int kw, const double sum) {
    const int w = seg * c.L + kw;
    if (kw >= 0 && kw < c.L && w < c.nWt) {
        const unsigned a = c.ctab + (unsigned)(w * 8);
        sts64(a, lds64(a) + sum);
    }
}

// The MB completed window sums of every lane sit in part[slot][lane]; sum them over the lanes of
// each segment in fixed order and add to the window table.  Up to two segments per warp (every
// st >= 31): lane = slot, one unrolled pass over the 32 lanes split at `split`.  Otherwise one
// (segment, slot) task per lane and round.
template <int MB>
__device__ __forceinline__ void reduce_block(const EmitCtx& c, const int kw0, const int lane) {
    __syncwarp();
    if (c.ng == 1) {
        if (lane < MB) {
            const unsigned pr = c.part + (unsigned)(lane * kPartPitch * 8);
            double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
#pragma unroll
            for (int q = 0; q < 32; q += 4) {
                a0 += lds64(pr + 8 * q);
                a1 += lds64(pr + 8 * q + 8);
                a2 += lds64(pr + 8 * q + 16);
                a3 += lds64(pr + 8 * q + 24);
            }
            ctab_add(c, c.seg_first, kw0 + lane, (a0 + a1) + (a2 + a3));
        }
    } else if (c.ng == 2) {
        if (lane < MB) {
            const unsigned pr = c.part + (unsigned)(lane * kPartPitch * 8);
            double a0 = 0.0, a1 = 0.0, b0 = 0.0, b1 = 0.0;
#pragma unroll
            for (int q = 0; q < 32; q += 2) {
                const double v0 = lds64(pr + 8 * q), v1 = lds64(pr + 8 * q + 8);
                a0 += q < c.split ? v0 : 0.0;
                b0 += q < c.split ? 0.0 : v0;
                a1 += q + 1 < c.split ? v1 : 0.0;
                b1 += q + 1 < c.split ? 0.0 : v1;
            }
            ctab_add(c, c.seg_first, kw0 + lane, a0 + a1);
            ctab_add(c, c.seg_first + 1, kw0 + lane, b0 + b1);
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
            ctab_add(c, seg, kw0 + sl, s0 + s1);
        }
    }
    __syncwarp();
}

// One item: march `nblk` blocks of MB rows.  `xp` points at this lane's X value of the first row;
// rows >= rows_valid read as 0.  Each lane streams its column through a private FIFO in shared
// memory filled by 8-byte cp.async copies (kFifoBatches batches of PF rows in flight, so L2 / DRAM
// latency never reaches the FMAs); after every block of MB rows the MB completed window sums are
// reduced over the lanes of each segment.
template <int MB>
__device__ __forceinline__ void march(const double* __restrict__ xp, const double* __restrict__ xsafe,
                                      const int st, const int rows_valid, const int nblk,
                                      const double (&T)[MB], const int lane, const EmitCtx& c) {
    constexpr int PF = PfRows<MB>::v;
    static_assert(MB % PF == 0 && kFifoBatches * PF <= kFifoRows, "FIFO geometry");
    double acc[MB], xr[PF];
#pragma unroll
    for (int u = 0; u < MB; ++u) acc[u] = 0.0;
    const unsigned fl = c.fifo + (unsigned)(lane * 8);
    int row_pf = 0;                                // row index the next copy belongs to
#pragma unroll
    for (int k = 0; k < kFifoBatches; ++k) {
#pragma unroll
        for (int u = 0; u < PF; ++u) {
            const bool ok = row_pf < rows_valid;
            cp_async8(fl + (unsigned)((k * PF + u) * 256), ok ? xp : xsafe, ok);
            xp += st;
            ++row_pf;
        }
        cp_async_commit();
    }
    int fb = 0;                                    // FIFO batch holding the rows consumed next
    const unsigned pl = c.part + (unsigned)(lane * 8);
#pragma unroll 1
    for (int blk = 0; blk < nblk; ++blk) {
#pragma unroll
        for (int u = 0; u < MB; ++u) {
            if (u % PF == 0) {
                cp_async_wait<kFifoBatches - 1>();
                const unsigned fa = fl + (unsigned)(fb * PF * 256);
#pragma unroll
                for (int k = 0; k < PF; ++k) xr[k] = lds64(fa + k * 256);
#pragma unroll
                for (int k = 0; k < PF; ++k) {
                    const bool ok = row_pf < rows_valid;
                    cp_async8(fa + k * 256, ok ? xp : xsafe, ok);
                    xp += st;
                    ++row_pf;
                }
                cp_async_commit();
                fb = fb + 1 == kFifoBatches ? 0 : fb + 1;
            }
            const double x = xr[u % PF];
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
    cp_async_wait<0>();
}

__device__ __forceinline__ double tmpl_lerp(const double* __restrict__ tm, int n_tmpl, int j, double tscale) {
    const double u = ((double)j + 0.5) * tscale;
    int k = (int)u;                                   // u >= 0: truncation == floor
    k = k > n_tmpl - 2 ? n_tmpl - 2 : k;
    const double fr = u - (double)k;
    const double t0 = tm[k];
    return t0 + fr * (tm[k + 1] - t0);
}

// All items (32 flat (segment, column) slots each) and tap blocks of one window tile, one pass.
template <int MB>
__device__ __forceinline__ void run_tile(const int n, const int n_tmpl, const RGeom& q,
                                         const double* __restrict__ tm, const double* __restrict__ x,
                                         const bool square, const int lane, const int nseg, const int L,
                                         const int nWt, const int k0, const unsigned part,
                                         const unsigned fifo, const unsigned ctab) {
    EmitCtx c;
    c.slots = nseg * q.st; c.st = q.st; c.L = L; c.nWt = nWt;
    c.ctab = ctab; c.part = part; c.fifo = fifo;
    const int items = (c.slots + 31) >> 5;
    const int nblk = (L + MB - 1 + MB - 1) / MB;
    const long long lim = (long long)n + q.D;          // x entries >= lim are never needed
    for (int item = 0; item < items; ++item) {
        c.f0 = item << 5;
        c.seg_first = c.f0 / q.st;
        c.ng = min(c.f0 + 31, c.slots - 1) / q.st - c.seg_first + 1;
        c.split = c.ng == 1 ? 32 : (c.seg_first + 1) * q.st - c.f0;
        const int f = c.f0 + lane;
        const bool active = f < c.slots;
        const int seg = active ? f / q.st : 0;
        const int col = active ? f - seg * q.st : 0;
        for (int b = 0; b < q.nmb; ++b) {
            double T[MB];
#pragma unroll
            for (int m = 0; m < MB; ++m) {
                const long long j = (long long)(b * MB + m) * q.st + col;
                double g = 0.0;
                if (active && j < q.D) g = tmpl_lerp(tm, n_tmpl, (int)j, q.tscale);
                T[m] = square ? g * g : g;
            }
            const long long ebase = ((long long)(k0 + seg * L) + (long long)b * MB) * q.st + col;
            int rows_valid = 0;
            if (active && ebase < lim) {
                const long long rv = (lim - ebase + q.st - 1) / q.st;
                rows_valid = rv > (long long)nblk * MB ? nblk * MB : (int)rv;
            }
            march<MB>(x + (active ? ebase : 0), x, q.st, rows_valid, nblk, T, lane, c);
        }
    }
}

template <bool UNIFORM>
__global__ void __launch_bounds__(kRT, 3) k_chi2_ring(TileArgs a) {
    extern __shared__ double dsm[];                 // per warp: [kMBMax][kPartPitch] emit buffer, window table
    __shared__ __align__(16) double s_tmpl[kTmplSmem];
    __shared__ __align__(8) unsigned long long s_mbar;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
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
    __syncthreads();
    if (tma_ok) {
        const unsigned mb = (unsigned)__cvta_generic_to_shared(&s_mbar);
        unsigned done = 0;
        while (!done) {
            asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\nselp.u32 %0, 1, 0, p;\n}"
                         : "=r"(done) : "r"(mb) : "memory");
        }
    }
    // ---- from here on every warp works alone on its own trial ------------------------------------
    const long long trial = (long long)blockIdx.x * kRW + warp;
    if (trial >= (long long)a.tile * a.n_dur) return;
    const int pl = (int)(trial / a.n_dur), jd = (int)(trial - (long long)pl * a.n_dur);
    const DurEntry e = a.durtab[trial];
    Partial* out = a.partial + trial;
    if (e.skip || e.stride < a.dbg_min_st || e.stride > a.dbg_max_st) {
        if (lane == 0) { out->valid = 0; out->dchi2 = 0.0; out->depth = 0.0; out->start = 0; }
        return;
    }
    (void)jd;
    RGeom q;
    q.D = e.D; q.st = e.stride;
    q.nW = (a.n + q.st - 1) / q.st;
    q.M = (q.D + q.st - 1) / q.st;
    pick_mb(q.M, q.MB, q.nmb);
    q.Kt = UNIFORM ? kCW : kCW / 2;
    q.tscale = __ddiv_rn((double)(a.n_tmpl - 1), (double)q.D);
    const double* __restrict__ tm = tmpl_in_smem ? s_tmpl : a.tmpl;
    const double* __restrict__ x1 = a.x1 + (long long)pl * a.pitch;
    const double* __restrict__ x0 = a.x0 + (long long)pl * a.pitch;
    const double* __restrict__ s1 = a.s1 + (long long)pl * a.spitch;
    const double* __restrict__ s0 = a.s0 + (long long)pl * a.spitch;
    const double G_u = a.w_uniform * e.gg2;
    const double den_u = ((double)q.D * a.w_uniform) * e.gbar;
    double* const wsm = dsm + warp * kWarpSmem;
    const unsigned part = (unsigned)__cvta_generic_to_shared(wsm);
    const unsigned fifo = part + (unsigned)(kMBMax * kPartPitch * 8);
    double* const ctab = wsm + kMBMax * kPartPitch + kFifoRows * 32;
    const unsigned ctab_s = (unsigned)__cvta_generic_to_shared(ctab);
    Cand best; best.has = 0; best.d = 0.0; best.s = 0; best.depth = 0.0;

    for (int k0 = 0; k0 < q.nW; k0 += q.Kt) {
        const int nWt = min(q.Kt, q.nW - k0);
        // ---- segment count: minimise items * rows per item (one warp runs them all) -------------------
        int bc = 0x7fffffff, bn = 1;
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            const int ns = lane + 1 + 32 * r;
            if (ns <= nWt) {
                const int L = (nWt + ns - 1) / ns;
                const int items = (ns * q.st + 31) >> 5;
                const int cost = items * (((L + 2 * q.MB - 2) / q.MB) * q.MB + 8);
                if (cost < bc) { bc = cost; bn = ns; }
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const int oc = __shfl_xor_sync(0xffffffffu, bc, o), on = __shfl_xor_sync(0xffffffffu, bn, o);
            if (oc < bc || (oc == bc && on < bn)) { bc = oc; bn = on; }
        }
        const int nseg = bn;
        const int L = (nWt + nseg - 1) / nseg;
        for (int i = lane; i < (UNIFORM ? nWt : 2 * q.Kt); i += 32) ctab[i] = 0.0;
        __syncwarp();

        for (int pass = 0; pass < (UNIFORM ? 1 : 2); ++pass) {
            const double* __restrict__ x = pass == 0 ? x1 : x0;
            const unsigned ct = ctab_s + (unsigned)(pass * q.Kt * 8);
            switch (q.MB) {
                case 21: run_tile<21>(a.n, a.n_tmpl, q, tm, x, pass == 1, lane, nseg, L, nWt, k0, part, fifo, ct); break;
                case 16: run_tile<16>(a.n, a.n_tmpl, q, tm, x, pass == 1, lane, nseg, L, nWt, k0, part, fifo, ct); break;
                case 12: run_tile<12>(a.n, a.n_tmpl, q, tm, x, pass == 1, lane, nseg, L, nWt, k0, part, fifo, ct); break;
                case 8: run_tile<8>(a.n, a.n_tmpl, q, tm, x, pass == 1, lane, nseg, L, nWt, k0, part, fifo, ct); break;
                default: run_tile<4>(a.n, a.n_tmpl, q, tm, x, pass == 1, lane, nseg, L, nWt, k0, part, fifo, ct); break;
            }
        }
        __syncwarp();
        // ---- a5 + a8 per window of the tile, four windows per lane in flight ---------------------------
        for (int w0 = 0; w0 < nWt; w0 += 128) {
            double hi1[4], lo1[4], hi0[4], lo0[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int w = w0 + 32 * u + lane;
                const int sidx = (k0 + w) * q.st;
                const bool ok = w < nWt;
                hi1[u] = ok ? __ldg(s1 + sidx + q.D) : 0.0;
                lo1[u] = ok ? __ldg(s1 + sidx) : 0.0;
                if (!UNIFORM) {
                    hi0[u] = ok ? __ldg(s0 + sidx + q.D) : 1.0;
                    lo0[u] = ok ? __ldg(s0 + sidx) : 0.0;
                }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int w = w0 + 32 * u + lane;
                if (w < nWt) {
                    const int sidx = (k0 + w) * q.st;
                    const double swr = hi1[u] - lo1[u];
                    const double den = UNIFORM ? den_u : (hi0[u] - lo0[u]) * e.gbar;
                    // a = max(rbar, 0) / mean(g_D),  rbar = swr / sw   (one division)
                    const double depth = __ddiv_rn(fmax(swr, 0.0), den);
                    const double C = ctab[w];
                    const double Gv = UNIFORM ? G_u : ctab[q.Kt + w];
                    const double d = -2.0 * depth * C + (depth * depth) * Gv;
                    cand_offer(best, d, sidx, depth);
                }
            }
        }
        __syncwarp();
    }

    // warp-wide lexicographic min on (d, s)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        Cand c;
        c.d = __shfl_xor_sync(0xffffffffu, best.d, o);
        c.depth = __shfl_xor_sync(0xffffffffu, best.depth, o);
        c.s = __shfl_xor_sync(0xffffffffu, best.s, o);
        c.has = __shfl_xor_sync(0xffffffffu, best.has, o);
        if (c.has) cand_offer(best, c.d, c.s, c.depth);
    }
    if (lane == 0) { out->valid = best.has; out->dchi2 = best.d; out->depth = best.depth; out->start = best.s; }
}

}  // namespace

void launch_chi2_ring(const TileArgs& a, cudaStream_t st) {
    const long long trials = (long long)a.tile * a.n_dur;
    const unsigned grid = (unsigned)((trials + kRW - 1) / kRW);
    const size_t sm = (size_t)(kRW * kWarpSmem) * sizeof(double);
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
