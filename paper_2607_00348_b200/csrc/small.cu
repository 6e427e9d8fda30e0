// Fused small-N path (gtls_opts.path = 1): steps a1-a8 for one (light curve, trial period) in ONE CTA,
// everything between the light curve and the period's best window staying in shared memory.
//
//   PAPER.md:185-264 (section 2.3) is the chain it fuses: fold (Eq. 10), sort by phase, wrap pad (Fig. 3),
//   running sums (Eq. 14), and for every duration and strided start (Eq. 18) the mean-matched depth
//   (Eq. 12-13) and chi2 = chi2_0 - 2 a C + a^2 G (Eq. 15 + 16), reduced to the
//   lexicographic minimum over (chi2, duration index, start).
//
// A work item is a (curve, period) pair of a batch of light curves (one curve for gtls_search, many for
// gtls_search_batch); persistent CTAs take items from a device-wide counter.  Per item:
//   1. fold in fp64 (one IEEE division), key = floor(phase 2^32) << 32 | index              -> smem
//   2. sort: counting sort on the top 11 key bits, then an exact rank inside every run of equal codes by
//      (key32, fp64 phase, index) -- a stable sort by phase, bit-exact, any phase distribution    -> smem
//   3. gather x1 = w r in phase order + wrap pad + zeros, block-wide inclusive scan S1            -> smem
//   4. chi2: the (duration, window class) units of the period are taken by the CTA's warps from a
//      shared-memory counter; a warp runs one unit as a shift-register ring march (chi2_ring.cu) whose
//      X values are read straight from the period's x1 in shared memory (no FIFO, no cp.async); the columns
//      of each completed window are summed through a small per-warp buffer into a 512-entry window table
//      (a time slice of every segment), which is scored in a coalesced pass, 32 windows per step, S1 from
//      shared memory (a5, a8)
//   5. per-period argmin over (dchi2, duration, start), t0 from the permutation                     -> HBM
// HBM traffic per item: t and w r of the curve (L2 resident) and 32 B of output.
//
// Limits (the host front end checks them and takes the general tiled path otherwise): dy uniform, no
// top_k / fp32 variant, n_dur <= 32, every window class stride <= 31 columns, and n small enough for
// x1 + S1 + the permutation in the 227 KB of a CTA (n <= ~8000).
#include <cstdio>

#include "gtls_internal.cuh"

namespace gtls {

namespace {

#ifdef GTLS_SMALL_PROF
__device__ unsigned long long g_prof[16];
#define PROF_T(v) const long long v = clock64()
#define PROF_ADD(k, dt) do { if ((threadIdx.x & 31) == 0) atomicAdd(&g_prof[k], (unsigned long long)(dt)); } while (0)
#else
#define PROF_T(v)
#define PROF_ADD(k, dt)
#endif

#ifndef GTLS_SMALL_THREADS
#define GTLS_SMALL_THREADS 384
#endif
constexpr int kSmThreads = GTLS_SMALL_THREADS;
constexpr int kSmWarps = kSmThreads / 32;
constexpr int kSmBinBits = 11;
constexpr int kSmBins = 1 << kSmBinBits;
constexpr int kSmPF = 8;                       // rows per batch of the march
constexpr int kSmPitch = 36;                   // doubles per row of the emit buffer
constexpr int kSmPart = kSmPF * kSmPitch;      // emit buffer doubles per warp (one batch: it is summed before the next one starts)
constexpr int kSmTab = 512;                    // window-table doubles per warp
constexpr int kSmMaxDur = 32;
constexpr int kSmTmpl = 512;

// window classes of a trial with M taps: rings of at most 24 taps (no narrow / wide distinction here)
__host__ __device__ __forceinline__ int sm_classes(int M) { return (M + 23) / 24; }

struct SmDur {             // one duration of the current period
    int D, st, ncls, skip;
    int unit0;             // index of its first (duration, class) unit
    int nW;                // trial starts
    double gbar, gg2;
};
struct SmCand { double d, depth; int s, has; };

__device__ __forceinline__ double lds64(const unsigned addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts64(const unsigned addr, const double v) {
    asm volatile("st.shared.f64 [%0], %1;" ::"r"(addr), "d"(v) : "memory");
}
__device__ __forceinline__ void offer(SmCand& b, const double d, const int s, const double depth) {
    if (!b.has || d < b.d || (d == b.d && s < b.s)) { b.d = d; b.s = s; b.depth = depth; b.has = 1; }
}
__device__ __forceinline__ double tmpl_lerp(const double* __restrict__ tm, int n_tmpl, int j, double tscale) {
    const double u = ((double)j + 0.5) * tscale;
    int k = (int)u;                                   // u >= 0: truncation == floor
    k = k > n_tmpl - 2 ? n_tmpl - 2 : k;
    const double fr = u - (double)k;
    const double t0 = tm[k];
    return t0 + fr * (tm[k + 1] - t0);
}

// One window class of one duration: windows kappa = 0 .. nWr-1 start at s = off + kappa * stp, the template
// index is j = m * stp + i (tap m < MB, column i < stp).  G = floor(32 / stp) segments of L consecutive
// windows sit side by side in the warp (one segment when stp > 16); lane = (segment, column).
struct SmCls {
    int n, D, stp, off, nWr;
    double G_u, inv_den;           // uniform dy: G = w sum g^2,  a = max(sum_W w r, 0) * inv_den
    unsigned xs, ss;               // shared-space addresses of x1 and S1 of the period
    int zidx;                      // index of a zero cell of x1 (reads beyond the pad are redirected to it)
    unsigned part;                 // this warp's emit buffer
    unsigned tab;                  // this warp's window table (kSmTab doubles)
    // debug instantiation only (gtls_ring_window_chi2 with path = 1): every window's dchi2 / depth by start / st0
    double* dbg_d; double* dbg_a; int st0;
};

// Template taps of one lane: g_D[m * stp + col] for m = m0 .. m0 + count - 1 (linear interpolation at the cell
// centres, reading G14) into the lane's column of the warp's emit buffer, 256 bytes per tap.  One copy of this
// code for every ring size (the kernel is bound by instruction fetch, not by arithmetic).
__device__ __noinline__ void sm_taps(const unsigned tl, const int m0, const int count, const int stp, const int col,
                                     const int D, const bool active, const double* __restrict__ tm, const int n_tmpl,
                                     const double tscale) {
#pragma unroll 2
    for (int m = 0; m < count; ++m) {
        const int j = (m0 + m) * stp + col;
        sts64(tl + (unsigned)(m * 256), (active && j < D) ? tmpl_lerp(tm, n_tmpl, j, tscale) : 0.0);
    }
}

// Score the windows of a table slice (a5 + a8): entry g * SL + o holds the in-transit sum C of the window
// that completed at row rho_base + o of segment g.  Coalesced over the table: 32 windows per step, every
// lane busy, four steps in flight.  Within a lane the starts ascend, so a strict '<' keeps the first of equal
// scores.  (One copy for every ring size: not inlined, everything passed by value.)
struct SmScore { unsigned tab, ss; int D, stp, off, nWr, G, L, lsl, kw_base, count; double G_u, inv_den; double* dbg_d; double* dbg_a; int st0; };
template <bool DBG>
__device__ __noinline__ SmCand sm_score_slice(const SmScore c, SmCand best, const int lane) {
    const int SL = 1 << c.lsl;
    double bd = best.has ? best.d : __longlong_as_double(0x7ff0000000000000LL), bdepth = best.depth;
    int bs = best.has ? best.s : -1;
    const int bs0 = bs;
#pragma unroll 1
    for (int i0 = 0; i0 < c.count; i0 += 128) {
        double C[4], hi[4], lo[4];
        int sidx[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int i = i0 + 32 * k + lane;
            const int g = i >> c.lsl, o = i & (SL - 1);
            const int kw = c.kw_base + o;
            const int kap = g * c.L + kw;
            const bool ok = g < c.G && kw >= 0 && kw < c.L && kap < c.nWr;
            const int sx = ok ? c.off + kap * c.stp : 0;
            sidx[k] = ok ? sx : -1;
            C[k] = lds64(c.tab + (unsigned)(i * 8));
            hi[k] = lds64(c.ss + (unsigned)((sx + c.D) * 8));
            lo[k] = lds64(c.ss + (unsigned)(sx * 8));
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const double swr = fmax(hi[k] - lo[k], 0.0);
            const double depth = swr * c.inv_den;
            const double d = -2.0 * depth * C[k] + (depth * depth) * c.G_u;
            if constexpr (DBG) { if (sidx[k] >= 0) { c.dbg_d[sidx[k] / c.st0] = d; c.dbg_a[sidx[k] / c.st0] = depth; } }
            // (a lane's previous best from an EARLIER class may have a later start: the lexicographic rule)
            const bool take = sidx[k] >= 0 && (d < bd || (d == bd && sidx[k] < bs));
            bd = take ? d : bd; bdepth = take ? depth : bdepth; bs = take ? sidx[k] : bs;
        }
    }
    if (bs != bs0 || bs >= 0) { best.d = bd; best.depth = bdepth; best.s = bs; best.has = bs >= 0 ? 1 : 0; }
    return best;
}

template <int MB, bool DBG>
__device__ __forceinline__ void sm_march(const SmCls& c, const double* __restrict__ tm, const int n_tmpl,
                                         const double tscale, const int lane, SmCand& best) {
    constexpr int PF = kSmPF, XQ = 4, LA = 3;
    const int G = c.stp <= 16 ? 32 / c.stp : 1;
    const int L = (c.nWr + G - 1) / G;
    const bool active = lane < G * c.stp;
    const int seg = min(lane / c.stp, G - 1);
    const int col = lane - seg * c.stp;
    // taps: computed in a rolled loop (the interpolation is ~25 instructions per tap) into this lane's
    // column of the still unused emit buffer, 12 at a time, then loaded into registers
    double T[MB];
    {
        const unsigned tl = c.tab + (unsigned)(lane * 8);       // (the window table is not in use yet)
#pragma unroll
        for (int h = 0; h < MB; h += 12) {
            constexpr int kHalf = 12;
            sm_taps(tl, h, min(kHalf, MB - h), c.stp, col, c.D, active, tm, n_tmpl, tscale);
#pragma unroll
            for (int m = h; m < h + kHalf; ++m)
                if (m < MB) T[m] = lds64(tl + (unsigned)((m - h) * 256));
        }
    }
    double acc[MB + 1], xq[XQ];
#pragma unroll
    for (int u = 0; u <= MB; ++u) acc[u] = 0.0;
    const int nbat = (L + MB - 1 + PF - 1) / PF;
    int e = c.off + seg * L * c.stp + col;         // x1 index of this lane's value of the next row to read
    if (!active) e = c.zidx;
#pragma unroll
    for (int k = 0; k < LA; ++k) { xq[k] = lds64(c.xs + (unsigned)(min(e, c.zidx) * 8)); e += c.stp; }

    // window table: a time slice of SL rows for each of the G segments (SL a power of two)
    int lg = 0;
    while ((1 << lg) < G) ++lg;
    int lsl = 9 - lg;                              // kSmTab = 512 entries
    while (lsl > 3 && (1 << (lsl - 1)) >= nbat * PF) --lsl;      // short marches: a smaller slice, fewer entries to score
    const int SL = 1 << lsl;
    // (stp >= 2 here: stride-1 classes take sm_march_direct)
    const unsigned pcur = c.part + (unsigned)(lane * 8);
    int rho_base = 0;
    // column sums of a batch: a task = (segment g, window slot sl); R lanes per task, each adding at most four
    // consecutive columns of the emit buffer, then log2(R) shuffle steps.  stp >= 2 means at most four rounds
    // of 32 / R tasks; what a lane does in round k never changes, so its addresses are set up once here.
    const int R = c.stp <= 4 ? 1 : (c.stp <= 8 ? 2 : (c.stp <= 16 ? 4 : 8));
    const int ntask = G * PF, tpr = 32 / R;
    const int nround = (ntask + tpr - 1) / tpr;          // <= 4
    const int r4 = (lane % R) * 4;
    unsigned rsrc[4];                                    // emit-buffer address of the lane's first column
    int rdst[4], rleft[4];                               // table offset (or -1), columns to add (0 .. 4)
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int task = k * tpr + lane / R;
        const bool tv = task < ntask;
        const int g = tv ? task / PF : 0, sl = task % PF;
        rsrc[k] = c.part + (unsigned)((sl * kSmPitch + g * c.stp + r4) * 8);
        rleft[k] = tv ? min(max(c.stp - r4, 0), 4) : 0;
        rdst[k] = (tv && r4 == 0) ? ((g << lsl) + sl) * 8 : -1;
    }
    SmScore sc;
    sc.tab = c.tab; sc.ss = c.ss; sc.D = c.D; sc.stp = c.stp; sc.off = c.off; sc.nWr = c.nWr; sc.G = G; sc.L = L; sc.lsl = lsl;
    sc.G_u = c.G_u; sc.inv_den = c.inv_den; sc.dbg_d = c.dbg_d; sc.dbg_a = c.dbg_a; sc.st0 = c.st0;
    sc.count = min(kSmTab, G << lsl);              // table entries in use
    __syncwarp();

#pragma unroll 1
    for (int b = 0; b < nbat; ++b) {
        PROF_T(pt0);
#pragma unroll
        for (int u = 0; u < PF; ++u) {
            xq[(u + LA) % XQ] = lds64(c.xs + (unsigned)(min(e, c.zidx) * 8));
            e += c.stp;
            const double xv = xq[u % XQ];
#pragma unroll
            for (int m = MB - 1; m >= 1; --m) acc[m + 1] = fma(T[m], xv, acc[m]);
            acc[1] = T[0] * xv;
            sts64(pcur + (unsigned)(u * kSmPitch * 8), acc[MB]);
        }
        __syncwarp();
        PROF_T(pt1);
        PROF_ADD(4, pt1 - pt0);
        const int o0 = b * PF - rho_base;          // table column of the batch's first row
        const unsigned tb = c.tab + (unsigned)(o0 * 8);
        // two rounds at a time, their loads first: the shared-memory accesses are volatile asm statements that the
        // compiler keeps in order, so a store between two rounds' loads serialises their latencies
#pragma unroll
        for (int k0 = 0; k0 < 4; k0 += 2) {
            if (k0 < nround) {                     // (warp uniform)
                double q[2][4], v[2];
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int k = k0 + h;
                    q[h][0] = rleft[k] > 0 ? lds64(rsrc[k]) : 0.0;
                    q[h][1] = rleft[k] > 1 ? lds64(rsrc[k] + 8) : 0.0;
                    q[h][2] = rleft[k] > 2 ? lds64(rsrc[k] + 16) : 0.0;
                    q[h][3] = rleft[k] > 3 ? lds64(rsrc[k] + 24) : 0.0;
                }
#pragma unroll
                for (int h = 0; h < 2; ++h) v[h] = (q[h][0] + q[h][1]) + (q[h][2] + q[h][3]);
                if (R >= 2) { v[0] += __shfl_xor_sync(0xffffffffu, v[0], 1); v[1] += __shfl_xor_sync(0xffffffffu, v[1], 1); }
                if (R >= 4) { v[0] += __shfl_xor_sync(0xffffffffu, v[0], 2); v[1] += __shfl_xor_sync(0xffffffffu, v[1], 2); }
                if (R >= 8) { v[0] += __shfl_xor_sync(0xffffffffu, v[0], 4); v[1] += __shfl_xor_sync(0xffffffffu, v[1], 4); }
#pragma unroll
                for (int h = 0; h < 2; ++h)
                    if (rdst[k0 + h] >= 0) sts64(tb + (unsigned)rdst[k0 + h], v[h]);
            }
        }
        __syncwarp();                              // the emit buffer is free for the next batch
        PROF_T(pt2);
        PROF_ADD(5, pt2 - pt1);
        if (o0 + PF == SL || b == nbat - 1) {      // the slice is full (or the march ends): score and recycle it
            __syncwarp();
            sc.kw_base = rho_base - (MB - 1);
            best = sm_score_slice<DBG>(sc, best, lane);
            __syncwarp();
            rho_base += SL;
            PROF_T(pt3);
            PROF_ADD(6, pt3 - pt2);
        }
    }
}

// Stride-1 classes (stp == 1: every start is a trial position, D <= 24): the lane's ring value IS the window sum,
// so each row's completed window is scored in place (a5, a8) -- no emit buffer, no table.  32 segments of L
// consecutive windows, L odd so that the lanes' x1 / S1 reads (L doubles apart) do not share banks; within a
// lane the starts ascend, so a strict '<' keeps the first of equal scores.
template <int MB, bool DBG>
__device__ __forceinline__ void sm_march_direct(const SmCls& c, const double* __restrict__ tm, const int n_tmpl,
                                                const double tscale, const int lane, SmCand& best) {
    constexpr int PF = kSmPF, XQ = 4, LA = 3;
    const int L = ((c.nWr + 31) / 32) | 1;
    double T[MB];
    {
        const unsigned tl = c.tab + (unsigned)(lane * 8);       // (the window table is not in use yet)
#pragma unroll
        for (int h = 0; h < MB; h += 12) {
            sm_taps(tl, h, min(12, MB - h), 1, 0, c.D, true, tm, n_tmpl, tscale);
#pragma unroll
            for (int m = h; m < h + 12; ++m)
                if (m < MB) T[m] = lds64(tl + (unsigned)((m - h) * 256));
        }
    }
    double acc[MB + 1], xq[XQ];
#pragma unroll
    for (int u = 0; u <= MB; ++u) acc[u] = 0.0;
    const int nbat = (L + MB - 1 + PF - 1) / PF;
    const int k0 = lane * L;                       // first window of this lane's segment (s = off + kappa, off = 0)
    int e = c.off + k0;
#pragma unroll
    for (int k = 0; k < LA; ++k) { xq[k] = lds64(c.xs + (unsigned)(min(e, c.zidx) * 8)); ++e; }
    // S1 at the start / end of the window that completes at row rho: S1[k0 + rho - (MB-1)] and the same + D;
    // clamped below for the warm-up rows (their windows are not scored)
    double bd = __longlong_as_double(0x7ff0000000000000LL), bdepth = 0.0;
    int bs = -1;
#pragma unroll 1
    for (int b = 0; b < nbat; ++b) {
#pragma unroll
        for (int u = 0; u < PF; ++u) {
            xq[(u + LA) % XQ] = lds64(c.xs + (unsigned)(min(e, c.zidx) * 8));
            ++e;
            const int kw = b * PF + u - (MB - 1);
            const int kap = k0 + kw;
            const bool ok = kw >= 0 && kw < L && kap < c.nWr;
            const int s = ok ? c.off + kap : 0;
            const double hi = lds64(c.ss + (unsigned)((s + c.D) * 8)), lo = lds64(c.ss + (unsigned)(s * 8));
            const double xv = xq[u % XQ];
#pragma unroll
            for (int m = MB - 1; m >= 1; --m) acc[m + 1] = fma(T[m], xv, acc[m]);
            acc[1] = T[0] * xv;
            const double swr = fmax(hi - lo, 0.0);
            const double depth = swr * c.inv_den;
            const double d = -2.0 * depth * acc[MB] + (depth * depth) * c.G_u;
            if constexpr (DBG) { if (ok) { c.dbg_d[s / c.st0] = d; c.dbg_a[s / c.st0] = depth; } }
            const bool take = ok && d < bd;
            bd = take ? d : bd; bdepth = take ? depth : bdepth; bs = take ? s : bs;
        }
    }
    if (bs >= 0) offer(best, bd, bs, bdepth);
}

template <bool DBG>
__device__ __forceinline__ void sm_run_unit(const SmCls& c, const int taps, const double* __restrict__ tm,
                                            const int n_tmpl, const double tscale, const int lane, SmCand& best) {
    // few ring sizes: the instruction cache, not the FP64 pipe, is what this kernel runs out of (twelve
    // warps in different phases of different bodies), so a ring is allowed to be up to twice its taps
    if (c.stp == 1) {
        if (taps > 12) sm_march_direct<24, DBG>(c, tm, n_tmpl, tscale, lane, best);
        else sm_march_direct<12, DBG>(c, tm, n_tmpl, tscale, lane, best);
        return;
    }
    if (taps > 16) sm_march<24, DBG>(c, tm, n_tmpl, tscale, lane, best);
    else if (taps > 8) sm_march<16, DBG>(c, tm, n_tmpl, tscale, lane, best);
    else sm_march<8, DBG>(c, tm, n_tmpl, tscale, lane, best);
}

// strict total order (key32, fp64 phase, index) == (fp64 phase, index)
__device__ __noinline__ bool sm_key_less(const u64 a, const u64 b, const double* __restrict__ t, const double period) {
    const u32 ka = (u32)(a >> 32), kb = (u32)(b >> 32);
    if (ka != kb) return ka < kb;
    const double pa = fold_phase(t[(u32)a], period), pb = fold_phase(t[(u32)b], period);
    if (pa != pb) return pa < pb;
    return (u32)a < (u32)b;
}

template <bool DBG>
__global__ void __launch_bounds__(kSmThreads, 1) k_tls_small(SmallArgs a) {
    extern __shared__ __align__(16) unsigned char sm_raw[];
    double* const xs = reinterpret_cast<double*>(sm_raw);                       // [a.xs_len]  (keysB during the sort)
    double* const ss = xs + a.xs_len;                                           // [a.xs_len]  (keysA during the sort)
    double* const part = ss + a.xs_len;                                         // [kSmWarps][kSmPart]
    double* const tabs = part + kSmWarps * kSmPart;                             // [kSmWarps][kSmTab]
    double* const tmpl_s = tabs + kSmWarps * kSmTab;                            // [kSmTmpl]
    SmCand* const wbest = reinterpret_cast<SmCand*>(tmpl_s + kSmTmpl);          // [kSmWarps][kSmMaxDur]
    SmDur* const dur = reinterpret_cast<SmDur*>(wbest + kSmWarps * kSmMaxDur);  // [kSmMaxDur]
    u32* const hist = reinterpret_cast<u32*>(dur + kSmMaxDur);                  // [kSmBins + 1]
    unsigned short* const perm = reinterpret_cast<unsigned short*>(hist + kSmBins + 8);   // [a.n_max]
    __shared__ __align__(8) unsigned long long s_mbar;
    __shared__ double s_scan[kSmWarps];
    __shared__ u32 s_wsum[kSmWarps];
    __shared__ long long s_item;
    __shared__ int s_next, s_units;
    u64* const keysA = reinterpret_cast<u64*>(ss);
    u64* const keysB = reinterpret_cast<u64*>(xs);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // ---- template nodes -> shared memory: one TMA bulk copy when size / alignment allow ------
    const bool tmpl_in_smem = a.n_tmpl <= kSmTmpl;
    const unsigned tbytes = (unsigned)a.n_tmpl * 8u;
    const bool tma_ok = tmpl_in_smem && (tbytes % 16u == 0) && (((unsigned long long)a.tmpl & 15ull) == 0);
    if (tma_ok) {
        const unsigned mb = (unsigned)__cvta_generic_to_shared(&s_mbar);
        if (tid == 0) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mb));
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mb), "r"(tbytes) : "memory");
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"((unsigned)__cvta_generic_to_shared(tmpl_s)), "l"(a.tmpl), "r"(tbytes), "r"(mb)
                         : "memory");
        }
    } else if (tmpl_in_smem) {
        for (int k = tid; k < a.n_tmpl; k += kSmThreads) tmpl_s[k] = a.tmpl[k];
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
    const double* __restrict__ tm = tmpl_in_smem ? tmpl_s : a.tmpl;

    int curve = 0;                                  // items come in (curve, period) order: the search moves forward
    for (;;) {
        if (tid == 0) s_item = (long long)atomicAdd(a.queue, 1ull);
        __syncthreads();
        const long long item = s_item;
        if (item >= a.n_items) break;
        PROF_T(k0);
        while (item >= a.per_off[curve + 1]) ++curve;
        const long long c0 = a.curve_off[curve];
        const int n = (int)(a.curve_off[curve + 1] - c0);
        const double* __restrict__ t = a.t + c0;
        const double* __restrict__ wr = a.wr + c0;
        const double period = a.periods[item];
        const double w_u = a.info[curve].w_min;
        const double chi2_0 = a.info[curve].chi2_0;
        const double* qrow = a.dur_per_period ? a.durs + item * (long long)a.n_dur : a.durs;

        // ---- durations of this period: D, stride, classes, template sums --------------------
        // (one L2 round trip for the fractions, one for the template sums; duplicates from shared memory)
        if (tid < a.n_dur) dur[tid].D = points_in_duration(qrow[tid], n);
        __syncthreads();
        SmDur e;
        e.D = 1; e.skip = 0;
        if (tid < a.n_dur) {
            e.D = dur[tid].D;
            e.gbar = __ddiv_rn(a.gtab[2 * e.D], (double)e.D);
            e.gg2 = a.gtab[2 * e.D + 1];
            for (int k = 0; k < tid; ++k) e.skip |= (dur[k].D == e.D);
            e.st = t0_stride(e.D, a.dt0);
            const int M = (e.D + e.st - 1) / e.st;
            e.ncls = e.skip ? 0 : sm_classes(M);
            e.nW = (n + e.st - 1) / e.st;
            e.unit0 = 0;
        }
        __syncthreads();                                // every D has been read before the records are written
        if (tid < a.n_dur) dur[tid] = e;
        for (int k = tid; k <= kSmBins; k += kSmThreads) hist[k] = 0;
        for (int k = tid; k < kSmWarps * kSmMaxDur; k += kSmThreads) wbest[k].has = 0;
        __syncthreads();
        int pad = 0;
        if (tid == 0) {
            int u = 0;
            for (int jd = 0; jd < a.n_dur; ++jd) { dur[jd].unit0 = u; u += dur[jd].ncls; }
            s_units = u;
            s_next = 0;
        }
        for (int jd = 0; jd < a.n_dur; ++jd) pad = max(pad, dur[jd].D);

        PROF_T(s0);
        PROF_ADD(8, s0 - k0);
        // ---- a1 fold + a2 sort ------------------------------------------------------------------
        // (t comes from the L2: two loads in flight per thread; the division is ~60 instructions, so no wider unroll)
        for (int i0 = 0; i0 < n; i0 += 2 * kSmThreads) {
            double tv[2];
#pragma unroll
            for (int k = 0; k < 2; ++k) { const int i = i0 + k * kSmThreads + tid; tv[k] = i < n ? t[i] : 0.0; }
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                const int i = i0 + k * kSmThreads + tid;
                if (i < n) {
                    const u32 k32 = phase_key32(fold_phase(tv[k], period));
                    atomicAdd(&hist[k32 >> (32 - kSmBinBits)], 1u);
                    keysA[i] = ((u64)k32 << 32) | (u64)(u32)i;
                }
            }
        }
        __syncthreads();
        PROF_T(s1);
        PROF_ADD(9, s1 - s0);
        {   // exclusive scan of the bin counts (kSmBins / kSmThreads per thread)
            constexpr int PER = (kSmBins + kSmThreads - 1) / kSmThreads;
            u32 cnt[PER], sum = 0;
#pragma unroll
            for (int k = 0; k < PER; ++k) { cnt[k] = tid * PER + k < kSmBins ? hist[tid * PER + k] : 0u; sum += cnt[k]; }
            u32 x = sum;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const u32 y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
            if (lane == 31) s_wsum[warp] = x;
            __syncthreads();
            u32 base = x - sum;
#pragma unroll
            for (int k = 0; k < kSmWarps; ++k) base += k < warp ? s_wsum[k] : 0u;
#pragma unroll
            for (int k = 0; k < PER; ++k) { if (tid * PER + k < kSmBins) hist[tid * PER + k] = base; base += cnt[k]; }
        }
        __syncthreads();
        PROF_T(s2);
        PROF_ADD(10, s2 - s1);
        for (int i = tid; i < n; i += kSmThreads) {            // scatter: any order inside a bin
            const u64 k = keysA[i];
            keysB[atomicAdd(&hist[(u32)(k >> 32) >> (32 - kSmBinBits)], 1u)] = k;
        }
        __syncthreads();                                        // hist[b] is now the END of bin b
        PROF_T(s3);
        PROF_ADD(11, s3 - s2);
        for (int i = tid; i < n; i += kSmThreads) {            // exact rank inside the bin
            const u64 k = keysB[i];
            const u32 bin = (u32)(k >> 32) >> (32 - kSmBinBits);
            const int rs = bin ? (int)hist[bin - 1] : 0, re = (int)hist[bin];
            int r = i;
            if (re - rs > 1) {
                r = rs;
                bool tie = false;
                for (int j = rs; j < re; ++j) {
                    const u64 o = keysB[j];
                    r += o < k ? 1 : 0;
                    tie |= j != i && (u32)(o >> 32) == (u32)(k >> 32);
                }
                if (tie) {                                      // equal 32-bit keys (rare): the fp64 phases decide
                    r = rs;
                    for (int j = rs; j < re; ++j) r += (j != i && sm_key_less(keysB[j], k, t, period)) ? 1 : 0;
                }
            }
            perm[r] = (unsigned short)(u32)k;
        }
        __syncthreads();
        PROF_T(s4);
        PROF_ADD(12, s4 - s3);
        // ---- a3 gather + wrap pad + zeros, a4 inclusive scan -----------------------------------
        const int len = n + pad;
        for (int i0 = 0; i0 < a.xs_len; i0 += 4 * kSmThreads) {       // four L2 loads in flight per thread
            double v[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) { const int i = i0 + k * kSmThreads + tid; v[k] = i < len ? wr[perm[i < n ? i : i - n]] : 0.0; }
#pragma unroll
            for (int k = 0; k < 4; ++k) { const int i = i0 + k * kSmThreads + tid; if (i < a.xs_len) xs[i] = v[k]; }
        }
        __syncthreads();
        PROF_T(s5);
        PROF_ADD(13, s5 - s4);
        {
            const int per = (len + kSmThreads - 1) / kSmThreads;
            const int i0 = min(len, tid * per), i1 = min(len, i0 + per);
            double sum = 0.0;
            for (int i = i0; i < i1; ++i) sum += xs[i];
            double x = sum;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const double y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
            if (lane == 31) s_scan[warp] = x;
            __syncthreads();
            double base = x - sum;
#pragma unroll
            for (int k = 0; k < kSmWarps; ++k) base += k < warp ? s_scan[k] : 0.0;
            if (tid == 0) ss[0] = 0.0;
            for (int i = i0; i < i1; ++i) { base += xs[i]; ss[i + 1] = base; }
        }
        __syncthreads();

        PROF_T(k1);
        PROF_ADD(0, k1 - k0);          // sort + scan phase (per warp)
        // ---- a5-a8: the (duration, class) units, longest durations first ------------------------
        {
            SmCls c;
            c.n = n;
            c.xs = (unsigned)__cvta_generic_to_shared(xs);
            c.ss = (unsigned)__cvta_generic_to_shared(ss);
            c.zidx = a.xs_len - 1;
            c.part = (unsigned)__cvta_generic_to_shared(part + warp * kSmPart);
            c.tab = (unsigned)__cvta_generic_to_shared(tabs + warp * kSmTab);
            const int units = s_units;
            for (;;) {
                int u = 0;
                if (lane == 0) u = atomicAdd(&s_next, 1);
                u = __shfl_sync(0xffffffffu, u, 0);
                if (u >= units) break;
                u = units - 1 - u;                              // long durations first (the tail is short units)
                int jd = a.n_dur - 1;
                while (dur[jd].unit0 > u || dur[jd].ncls == 0) --jd;
                const SmDur e = dur[jd];
                const int r = u - e.unit0;
                c.D = e.D; c.stp = e.ncls * e.st; c.off = r * e.st;
                c.nWr = e.nW > r ? (e.nW - r + e.ncls - 1) / e.ncls : 0;
                c.G_u = w_u * e.gg2;
                c.inv_den = __ddiv_rn(1.0, ((double)e.D * w_u) * e.gbar);
                SmCand best; best.has = 0; best.d = 0.0; best.s = 0; best.depth = 0.0;
                if (c.nWr > 0) {
                    const int taps = (e.D + c.stp - 1) / c.stp;
                    const double tscale = __ddiv_rn((double)(a.n_tmpl - 1), (double)e.D);
                    c.dbg_d = a.dbg_dchi2; c.dbg_a = a.dbg_depth; c.st0 = e.st;
                    sm_run_unit<DBG>(c, taps, tm, a.n_tmpl, tscale, lane, best);
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    SmCand o2;
                    o2.d = __shfl_xor_sync(0xffffffffu, best.d, o);
                    o2.depth = __shfl_xor_sync(0xffffffffu, best.depth, o);
                    o2.s = __shfl_xor_sync(0xffffffffu, best.s, o);
                    o2.has = __shfl_xor_sync(0xffffffffu, best.has, o);
                    if (o2.has) offer(best, o2.d, o2.s, o2.depth);
                }
                if (lane == 0 && best.has) {                    // this warp's best of duration jd so far
                    SmCand w = wbest[warp * kSmMaxDur + jd];
                    offer(w, best.d, best.s, best.depth);
                    wbest[warp * kSmMaxDur + jd] = w;
                }
                __syncwarp();
            }
        }
        PROF_T(k2);
        PROF_ADD(1, k2 - k1);          // busy in units
        __syncthreads();
        PROF_T(k3);
        PROF_ADD(2, k3 - k2);          // waiting for the slowest warp
        // ---- a8: per duration the best over the warps, then the first strict minimum over durations --
        if (warp == 0) {
            SmCand b; b.has = 0; b.d = 0.0; b.s = 0; b.depth = 0.0;
            if (lane < a.n_dur)
                for (int w = 0; w < kSmWarps; ++w) {
                    const SmCand o = wbest[w * kSmMaxDur + lane];
                    if (o.has) offer(b, o.d, o.s, o.depth);
                }
            int jd = lane;
            unsigned long long nwin = 0, npts = 0;
            if (lane < a.n_dur) {
                nwin = (unsigned long long)dur[lane].nW;
                npts = dur[lane].skip ? 0ull : nwin * (unsigned long long)dur[lane].D;
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const double od = __shfl_xor_sync(0xffffffffu, b.d, o);
                const double odep = __shfl_xor_sync(0xffffffffu, b.depth, o);
                const int os = __shfl_xor_sync(0xffffffffu, b.s, o);
                const int oh = __shfl_xor_sync(0xffffffffu, b.has, o);
                const int oj = __shfl_xor_sync(0xffffffffu, jd, o);
                if (oh && (!b.has || od < b.d || (od == b.d && oj < jd))) { b.d = od; b.depth = odep; b.s = os; b.has = 1; jd = oj; }
                nwin += __shfl_xor_sync(0xffffffffu, nwin, o);
                npts += __shfl_xor_sync(0xffffffffu, npts, o);
            }
            if (lane == 0) {
                if (!b.has) { jd = 0; b.d = 0.0; b.s = 0; b.depth = 0.0; }      // no usable window (reading G22)
                a.out_chi2[item] = chi2_0 + b.d;
                if (a.out_best) {
                    gtls_best o;
                    o.dur_idx = jd; o.start = b.s; o.depth = b.depth;
                    o.t0 = t[perm[(b.s + (dur[jd].D - 1) / 2) % n]];
                    a.out_best[item] = o;
                }
                atomicAdd(&a.counters[2 * curve], nwin);
                atomicAdd(&a.counters[2 * curve + 1], npts);
            }
        }
        __syncthreads();
    }
}

}  // namespace

#ifdef GTLS_SMALL_PROF
void small_prof_dump() {
    unsigned long long h[16];
    cudaMemcpyFromSymbol(h, g_prof, sizeof(h));
    fprintf(stderr, "small prof: sort %.3e units %.3e wait %.3e | rows %.3e reduce %.3e score %.3e\n", (double)h[0], (double)h[1], (double)h[2], (double)h[4], (double)h[5], (double)h[6]);
    fprintf(stderr, "  sort split: setup %.2e fold %.2e binscan %.2e scatter %.2e rank %.2e gather %.2e (scan = rest)\n", (double)h[8], (double)h[9], (double)h[10], (double)h[11], (double)h[12], (double)h[13]);
    unsigned long long z[16] = {};
    cudaMemcpyToSymbol(g_prof, z, sizeof(z));
}
#endif

size_t small_smem_bytes(int n_max, int d_max) {
    const size_t xs_len = ((size_t)n_max + d_max + 48 + 1) & ~(size_t)1;
    return 2 * xs_len * 8 + (size_t)kSmWarps * (kSmPart + kSmTab) * 8 + kSmTmpl * 8 + (size_t)kSmWarps * kSmMaxDur * sizeof(SmCand) +
           kSmMaxDur * sizeof(SmDur) + (kSmBins + 8) * sizeof(u32) + (((size_t)n_max * 2 + 15) & ~(size_t)15) + 64;
}

bool small_path_fits(int n_max, int d_max, int n_dur, double dt0) {
    if (n_max < 3 || n_max > 65535 || n_dur > kSmMaxDur) return false;
    if (small_smem_bytes(n_max, d_max) > 227u * 1024u - 256u) return false;
    for (int D = 1; D <= d_max; ++D) {                 // every class stride the grid can ask for
        const int st = dt0 > 0.0 ? ((int)((double)D * dt0) < 1 ? 1 : (int)((double)D * dt0)) : 1;
        const int M = (D + st - 1) / st;
        if (sm_classes(M) * st > 31) return false;
    }
    return true;
}

int launch_tls_small(SmallArgs& a, int n_max, int d_max, int sm_count, cudaStream_t st) {
    a.xs_len = (int)(((size_t)n_max + d_max + 48 + 1) & ~(size_t)1);
    a.n_max = n_max;
    const size_t sm = small_smem_bytes(n_max, d_max);
    long long grid = a.n_items < sm_count ? a.n_items : sm_count;
    if (a.dbg_dchi2) {             // gtls_ring_window_chi2 with path = 1: the instantiation that dumps every window's score
        cudaError_t e = cudaFuncSetAttribute(k_tls_small<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
        if (e != cudaSuccess) return (int)e;
        k_tls_small<true><<<(unsigned)grid, kSmThreads, sm, st>>>(a);
        return (int)cudaGetLastError();
    }
    cudaError_t e = cudaFuncSetAttribute(k_tls_small<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) return (int)e;
    k_tls_small<false><<<(unsigned)grid, kSmThreads, sm, st>>>(a);
#ifdef GTLS_SMALL_PROF
    cudaStreamSynchronize(st);
    small_prof_dump();
#endif
    return (int)cudaGetLastError();
}

}  // namespace gtls
