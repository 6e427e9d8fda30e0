// Steps a5-a8, in-transit chi2 as a register-ring correlation -- the dominant kernel.
//
// For one (period, duration) with D points per window and stride st between trial starts
// (Eq. 18), split the template index j = m*st + i (tap m < M = ceil(D/st),
// column i < st).  With the folded curve viewed as rows of st points, X[rho][i] = x1[rho*st+i],
//     C[k] = sum_i sum_m g[m*st+i] * X[k+m][i]                              (Eq. 16)
// is, per column i, a 1-D correlation along the rows with the M taps g[m*st+i].
//
// A lane owns ONE column and marches down its rows holding MB taps and a ring of MB window
// accumulators in registers: every X value is fetched from L2 exactly once and feeds MB DFMAs;
// each row step starts one window (DMUL) and completes one.  X is not staged as tiles: each lane
// streams its column through a private shared-memory FIFO filled by 8-byte cp.async copies issued
// ~20 rows ahead, so neither L2 nor DRAM latency reaches the FMAs and the FP64 pipe
// (64 DFMA/clk/SM) is the only busy resource.  Every PF rows the PF completed per-column sums of
// the 32 lanes are summed over the columns of a window in fixed order (deterministic) through a
// small per-warp buffer and land in the warp's window table.
//
// More than 21 taps never occur: a trial with M > 21 is split into c = ceil(M/21) window classes
// r = 0..c-1 (windows k = kappa*c + r), each of which is the same problem with stride c*st,
// ceil(D/(c*st)) <= 21 taps and the array shifted by r*st.
//
// ONE WARP OWNS ONE TRIAL (period, duration) from its first row to its argmin: there is no CTA
// barrier after the template nodes are staged, so the warps of an SM (6 CTAs x 2 warps) sit in different phases and
// the scoring of one hides behind the DFMAs of the others.
//   stride > 16 ("wide"): the columns are cut into ceil(stride/32) balanced chunks; the warp marches
//     one chunk at a time down the rows of a window tile (software-pipelined, march_pipe) and adds
//     its per-window sums into the table; windows are processed in tiles of the table size.
//   stride <= 16 ("narrow", short durations, very many windows): floor(32/stride) segments sit
//     side by side in the warp, the whole class is ONE march of ~n/32 rows, and the table is a
//     time slice that is scored and recycled every few blocks.
//
// a5 (depth from the prefix sums, Eq. 12-14), the score dchi2 = -2 a C + a^2 G (a6+a7; the
// S2 window term of Eq. 15 cancels against the same term of Eq. 16) and the lexicographic
// (dchi2, start) argmin (a8) run from the table.
// The template nodes are staged in shared memory with one TMA bulk copy (cp.async.bulk).
#include <cstdlib>

#include "gtls_internal.cuh"

namespace gtls {

namespace {

constexpr int kRT = 64;                  // threads per CTA (two trials: a CTA keeps its slot until both are done)
constexpr int kRW = kRT / 32;            // warps (= trials) per CTA
constexpr int kPartPitch = 36;           // doubles per slot row of the per-warp emit buffer
constexpr int kPartRows = 16;            // two emit buffers of max PfRows rows (pipelined column sums)
constexpr int kFifoBatches = 3;          // batches of PfRows rows per lane in the cp.async FIFO
constexpr int kFifoRows = 24;            // >= kFifoBatches * max PfRows
constexpr int kCW = 704;                 // window-table doubles per warp, narrow variants (>= 32 * 21)
constexpr int kCWWide = 2488;            // wide variants: window tiles of 2 460 windows (fewer warm-up rows, tap set-ups and FIFO primes
                                         // per trial).  Measured on c4, chi2 stage: 704 entries / 4 CTAs per SM 4.63 s, 1720 / 4: 4.61 s,
                                         // 2488 / 3: 4.52 s, 3128 / 3: 4.66 s (the tile's span outgrows what stays in the L2 between chunks)
constexpr int kTmplSmem = 512;           // template nodes cached in shared memory
constexpr unsigned kGridCap = 148u * 6u;   // CTAs per launch: the 6 resident CTAs per SM, persistent (dynamic trial queue)
constexpr unsigned kGridCapWide = 148u * 3u;
template <bool NARROW> struct WarpSmem { static constexpr int v = kPartRows * kPartPitch + kFifoRows * 32 + (NARROW ? kCW : kCWWide); };   // doubles per warp

struct Cand { double d; double depth; int s; int has; };

__device__ __forceinline__ void cand_offer(Cand& b, double d, int s, double depth) {
    if (!b.has || d < b.d || (d == b.d && s < b.s)) { b.d = d; b.s = s; b.depth = depth; b.has = 1; }
}

// rows per FIFO batch = completed windows reduced at once (divides MB)
template <int MB> struct PfRows { static constexpr int v = (MB % 7 == 0) ? 7 : (MB >= 16 ? 8 : (MB >= 8 ? MB / 2 : MB)); };

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
__device__ __forceinline__ void cp_async8(const unsigned dst, const double* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
}
// 16-byte copy (both addresses 16-byte aligned); `valid == false` writes zeros without reading
__device__ __forceinline__ void cp_async16(const unsigned dst, const double* src, const bool valid) {
    const int sz = valid ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// One window class of one trial, as seen by the owning warp.
struct Cls {
    int D, stp, off, nWr;                // window length, class stride, element offset, windows
    bool uniform;
    double G_u, inv_den_u, gbar;         // uniform dy: G and 1/(sw*gbar) are constants
    const double* s1; const double* s0;  // prefix sums of this period
    unsigned ctab;                       // shared-space address of the window table
    unsigned part;                       // shared-space address of the [kPartRows][kPartPitch] emit buffer
    unsigned fifo;                       // shared-space address of the [kFifoRows][32] X FIFO
    int Kt;                              // table entries per quantity (C, and G when dy is not uniform)
    // debug instantiation only (gtls_ring_window_chi2): every window's dchi2 / depth, indexed by start / st0
    double* dbg_d; double* dbg_a; int st0;
};

// a5 + a8 for one window kappa of the class (start s = off + kappa*stp): hi/lo are the prefix sums
// at s+D and s.  a = max(rbar, 0) / mean(g_D) with rbar = swr / sw.  Uniform dy: sw * mean(g_D) is a
// constant of the trial, so a = max(swr, 0) * inv_den (one multiply); otherwise one division.
template <bool DBG = false>
__device__ __forceinline__ void score_one(const Cls& c, Cand& best, const int s, const double hi1,
                                          const double lo1, const double hi0, const double lo0,
                                          const double C, const double Gt) {
    const double swr = fmax(hi1 - lo1, 0.0);
    const double depth = c.uniform ? swr * c.inv_den_u : __ddiv_rn(swr, (hi0 - lo0) * c.gbar);
    const double Gv = c.uniform ? c.G_u : Gt;
    const double d = -2.0 * depth * C + (depth * depth) * Gv;
    if constexpr (DBG) { c.dbg_d[s / c.st0] = d; c.dbg_a[s / c.st0] = depth; }
    if (d <= best.d || !best.has) cand_offer(best, d, s, depth);     // rarely taken after the first windows
}
// Wide path: score the windows [k0, k0 + nWt) of the class from table entries [0, nWt).
template <bool DBG = false>
__device__ __forceinline__ void score_wide(const Cls& c, Cand& best, const int lane, const int k0,
                                           const int nWt, const int toff) {
    for (int i0 = 0; i0 < nWt; i0 += 128) {
        double hi1[4], lo1[4], hi0[4], lo0[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int w = i0 + 32 * u + lane;
            const int s = c.off + (k0 + w) * c.stp;
            const bool ok = w < nWt;
            hi1[u] = ok ? __ldg(c.s1 + s + c.D) : 0.0;
            lo1[u] = ok ? __ldg(c.s1 + s) : 0.0;
            hi0[u] = 1.0; lo0[u] = 0.0;
            if (!c.uniform) {
                hi0[u] = ok ? __ldg(c.s0 + s + c.D) : 1.0;
                lo0[u] = ok ? __ldg(c.s0 + s) : 0.0;
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int w = i0 + 32 * u + lane;
            if (w < nWt) {
                const unsigned ta = c.ctab + (unsigned)((w + toff) * 8);
                score_one<DBG>(c, best, c.off + (k0 + w) * c.stp, hi1[u], lo1[u], hi0[u], lo0[u], lds64(ta),
                          c.uniform ? 0.0 : lds64(ta + (unsigned)(c.Kt * 8)));
            }
        }
    }
}

// Narrow path: table entry seg*SL + o holds window kw = kw_base + o of segment seg (kappa = seg*L + kw).
template <bool DBG = false>
__device__ __forceinline__ void score_narrow(const Cls& c, Cand& best, const int lane, const int G,
                                             const int SL, const int SLn, const float invSL,
                                             const int kw_base, const int L) {
    const int count = G * SL;
    for (int i0 = 0; i0 < count; i0 += 128) {
        double hi1[4], lo1[4], hi0[4], lo0[4];
        int sidx[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int i = i0 + 32 * u + lane;
            const int seg = (int)(((float)i + 0.5f) * invSL);
            const int o = i - seg * SL;
            const int kw = kw_base + o;
            const int kap = seg * L + kw;
            const bool ok = i < count && o < SLn && kw >= 0 && kw < L && kap < c.nWr;
            const int s = c.off + kap * c.stp;
            sidx[u] = ok ? s : -1;
            hi1[u] = ok ? __ldg(c.s1 + s + c.D) : 0.0;
            lo1[u] = ok ? __ldg(c.s1 + s) : 0.0;
            hi0[u] = 1.0; lo0[u] = 0.0;
            if (!c.uniform) {
                hi0[u] = ok ? __ldg(c.s0 + s + c.D) : 1.0;
                lo0[u] = ok ? __ldg(c.s0 + s) : 0.0;
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (sidx[u] >= 0) {
                const unsigned ta = c.ctab + (unsigned)((i0 + 32 * u + lane) * 8);
                score_one<DBG>(c, best, sidx[u], hi1[u], lo1[u], hi0[u], lo0[u], lds64(ta),
                          c.uniform ? 0.0 : lds64(ta + (unsigned)(c.Kt * 8)));
            }
        }
    }
}

struct It {                              // one march
    bool direct;                         // narrow with stride 1: no cross-lane sum
    int L;                               // windows per segment (wide: one segment = the window tile)
    int nWt;                             // wide: windows in the tile
    // narrow: G segments side by side, table slice of SL = KB*MB windows per segment
    int G, KB, SL, SLn;                  // SL = odd pitch >= SLn = KB*MB valid windows per segment
    float invSL;
    unsigned tab;                        // table of the quantity being accumulated (C or G)
};

__device__ __forceinline__ void tab_add(const unsigned a, const double v) { sts64(a, lds64(a) + v); }

// PF completed window sums per lane sit in part[slot][lane] (windows kwb .. kwb+PF-1 of the lane's
// segment): sum them over the lanes of each segment in fixed order.
template <int PF, bool NARROW>
__device__ __forceinline__ void reduce_batch(const Cls& c, const It& it, const int kwb, const int kw_base,
                                             const int lane) {
    __syncwarp();
    if constexpr (!NARROW) {
        // wide: the warp holds one segment; four lanes per slot, eight strided values each, two shuffle steps
        const int sl = lane >> 2, r = lane & 3;
        double v = 0.0;
        if (sl < PF) {
            const unsigned pr = c.part + (unsigned)((sl * kPartPitch + r) * 8);
            double a0 = 0.0, a1 = 0.0;
#pragma unroll
            for (int i = 0; i < 8; i += 2) { a0 += lds64(pr + 32 * i); a1 += lds64(pr + 32 * i + 32); }
            v = a0 + a1;
        }
        v += __shfl_xor_sync(0xffffffffu, v, 1);
        v += __shfl_xor_sync(0xffffffffu, v, 2);
        const int kw = kwb + sl;
        if (r == 0 && sl < PF && kw >= 0 && kw < it.L && kw < it.nWt) tab_add(it.tab + (unsigned)(kw * 8), v);
    } else {
        for (int t = lane; t < it.G * PF; t += 32) {
            const int g = t / PF, sl = t - g * PF;
            const unsigned pr = c.part + (unsigned)((sl * kPartPitch + g * c.stp) * 8);
            double a0 = 0.0, a1 = 0.0;
            int q = 0;
            for (; q + 1 < c.stp; q += 2) { a0 += lds64(pr + 8 * q); a1 += lds64(pr + 8 * q + 8); }
            if (q < c.stp) a0 += lds64(pr + 8 * q);
            sts64(it.tab + (unsigned)((g * it.SL + (kwb + sl - kw_base)) * 8), a0 + a1);
        }
    }
    __syncwarp();
}

// One march: `nblk` blocks of MB rows.  `xp` points at this lane's X value of the first row, rows
// >= rows_valid read as 0 (rows_min = the smallest rows_valid of the warp, so batches below it need
// no predicate).  Taps T[m] multiply row (window + m).  Narrow path: every KB blocks the table slice
// is scored and recycled.
template <int MB, bool NARROW, typename F, bool DBG = false>
__device__ __forceinline__ void march(const Cls& c, const It& it, const double* __restrict__ xp,
                                      const int rows_valid, const int rows_min, const int nblk,
                                      const F (&T)[MB], const int lane, Cand& best) {
    constexpr int PF = PfRows<MB>::v;
    static_assert(MB % PF == 0 && kFifoBatches * PF <= kFifoRows && PF <= kPartRows, "geometry");
    F acc[MB], xr[PF];
#pragma unroll
    for (int u = 0; u < MB; ++u) acc[u] = (F)0;
    const unsigned fl = c.fifo + (unsigned)(lane * 8);
    const long long rstride = (long long)c.stp;
    int row_pf = 0;                                // row index the next copy belongs to
#pragma unroll
    for (int k = 0; k < kFifoBatches; ++k) {
#pragma unroll
        for (int u = 0; u < PF; ++u) {
            cp_async8(fl + (unsigned)((k * PF + u) * 256), xp, row_pf < rows_valid);
            xp += rstride;
            ++row_pf;
        }
        cp_async_commit();
    }
    int fb = 0;                                    // FIFO batch holding the rows consumed next
    int kw_base = -(MB - 1), bis = 0;              // narrow: first window of the slice, blocks in it
    const unsigned part_lane = c.part + (unsigned)(lane * 8);
    const unsigned tab_lane = it.tab + (unsigned)(lane * it.SL * 8);
#pragma unroll 1
    for (int blk = 0; blk < nblk; ++blk) {
#pragma unroll
        for (int u = 0; u < MB; ++u) {
            if (u % PF == 0) {
                cp_async_wait<kFifoBatches - 1>();
                const unsigned fa = fl + (unsigned)(fb * PF * 256);
#pragma unroll
                for (int k = 0; k < PF; ++k) xr[k] = (F)lds64(fa + k * 256);
                if (row_pf + PF <= rows_min) {
#pragma unroll
                    for (int k = 0; k < PF; ++k) { cp_async8(fa + k * 256, xp); xp += rstride; }
                } else {
#pragma unroll
                    for (int k = 0; k < PF; ++k) { cp_async8(fa + k * 256, xp, row_pf + k < rows_valid); xp += rstride; }
                }
                row_pf += PF;
                cp_async_commit();
                fb = fb + 1 == kFifoBatches ? 0 : fb + 1;
            }
            const F x = xr[u % PF];
#pragma unroll
            for (int m = 0; m < MB; ++m) {
                const int a = (u - m + MB) % MB;
                if (m == 0) acc[a] = T[0] * x;                      // window gamma starts at this row
                else acc[a] = fma(T[m], x, acc[a]);
            }
            // window gamma - (MB-1) is complete
            const unsigned ea = (NARROW && it.direct) ? tab_lane + (unsigned)((bis * MB + u) * 8)
                                          : part_lane + (unsigned)((u % PF) * kPartPitch * 8);
            sts64(ea, (double)acc[(u + 1) % MB]);
            if (u % PF == PF - 1 && !(NARROW && it.direct))
                reduce_batch<PF, NARROW>(c, it, blk * MB + (u - (PF - 1)) - (MB - 1), kw_base, lane);
        }
        if (NARROW && ++bis == it.KB) {
            __syncwarp();
            score_narrow<DBG>(c, best, lane, it.G, it.SL, it.SLn, it.invSL, kw_base, it.L);
            __syncwarp();
            kw_base += it.SLn;
            bis = 0;
        }
    }
    cp_async_wait<0>();
    if (NARROW && bis > 0) {
        __syncwarp();
        score_narrow<DBG>(c, best, lane, it.G, it.SL, it.SLn, it.invSL, kw_base, it.L);
        __syncwarp();
    }
}

// Narrow path when dy is NOT uniform: C = sum g x1 and G = sum g^2 x0 are needed for every window of the
// time-sliced table, so both are accumulated in ONE march: two rings (C, G) over two FIFO streams
// (x1 = w r, x0 = w), taps g held once (g^2 x0 is taken as g * (g * x0)).  3 MB doubles of ring state:
// ring sizes up to 16.  Batches of kDualPF rows per stream, the two streams share the FIFO half and half;
// the emit buffer holds the C partials in rows [0, PF) and the G partials in rows [PF, 2 PF).
constexpr int kDualPF = 4;
template <int MB, typename F, bool DBG = false>
__device__ __forceinline__ void march_dual(const Cls& c, const It& it, const double* __restrict__ xp1,
                                           const double* __restrict__ xp0, const int rows_valid,
                                           const int rows_min, const int nblk, const F (&T)[MB],
                                           const int lane, Cand& best) {
    constexpr int PF = kDualPF;
    constexpr int kHalf = kFifoRows / 2;           // FIFO rows per stream
    static_assert(MB % PF == 0 && kFifoBatches * PF <= kHalf && 2 * PF <= kPartRows, "geometry");
    F accC[MB], accG[MB], xr1[PF], xr0[PF];
#pragma unroll
    for (int u = 0; u < MB; ++u) { accC[u] = (F)0; accG[u] = (F)0; }
    const unsigned fl1 = c.fifo + (unsigned)(lane * 8);
    const unsigned fl0 = fl1 + (unsigned)(kHalf * 256);
    const long long rstride = (long long)c.stp;
    int row_pf = 0;
#pragma unroll
    for (int k = 0; k < kFifoBatches; ++k) {
#pragma unroll
        for (int u = 0; u < PF; ++u) {
            cp_async8(fl1 + (unsigned)((k * PF + u) * 256), xp1, row_pf < rows_valid);
            cp_async8(fl0 + (unsigned)((k * PF + u) * 256), xp0, row_pf < rows_valid);
            xp1 += rstride; xp0 += rstride;
            ++row_pf;
        }
        cp_async_commit();
    }
    int fb = 0;
    int kw_base = -(MB - 1), bis = 0;
    const unsigned part_lane = c.part + (unsigned)(lane * 8);
    const unsigned tab_lane = it.tab + (unsigned)(lane * it.SL * 8);
    const unsigned gofs = (unsigned)(c.Kt * 8);    // G table behind the C table
#pragma unroll 1
    for (int blk = 0; blk < nblk; ++blk) {
#pragma unroll
        for (int u = 0; u < MB; ++u) {
            if (u % PF == 0) {
                cp_async_wait<kFifoBatches - 1>();
                const unsigned fa1 = fl1 + (unsigned)(fb * PF * 256), fa0 = fl0 + (unsigned)(fb * PF * 256);
#pragma unroll
                for (int k = 0; k < PF; ++k) { xr1[k] = (F)lds64(fa1 + k * 256); xr0[k] = (F)lds64(fa0 + k * 256); }
#pragma unroll
                for (int k = 0; k < PF; ++k) {
                    const bool ok = row_pf + k < rows_valid;
                    cp_async8(fa1 + k * 256, xp1, ok);
                    cp_async8(fa0 + k * 256, xp0, ok);
                    xp1 += rstride; xp0 += rstride;
                }
                row_pf += PF;
                cp_async_commit();
                fb = fb + 1 == kFifoBatches ? 0 : fb + 1;
            }
            const F x1v = xr1[u % PF], x0v = xr0[u % PF];
#pragma unroll
            for (int m = 0; m < MB; ++m) {
                const int a = (u - m + MB) % MB;
                const F gx = T[m] * x0v;
                if (m == 0) { accC[a] = T[0] * x1v; accG[a] = T[0] * gx; }
                else { accC[a] = fma(T[m], x1v, accC[a]); accG[a] = fma(T[m], gx, accG[a]); }
            }
            // window gamma - (MB-1) is complete
            if (it.direct) {
                const unsigned ea = tab_lane + (unsigned)((bis * MB + u) * 8);
                sts64(ea, (double)accC[(u + 1) % MB]);
                sts64(ea + gofs, (double)accG[(u + 1) % MB]);
            } else {
                const unsigned ea = part_lane + (unsigned)((u % PF) * kPartPitch * 8);
                sts64(ea, (double)accC[(u + 1) % MB]);
                sts64(ea + (unsigned)(PF * kPartPitch * 8), (double)accG[(u + 1) % MB]);
                if (u % PF == PF - 1) {
                    const int kwb = blk * MB + (u - (PF - 1)) - (MB - 1);
                    __syncwarp();
                    for (int t = lane; t < it.G * PF; t += 32) {
                        const int g = t / PF, sl = t - g * PF;
                        const unsigned pr = c.part + (unsigned)((sl * kPartPitch + g * c.stp) * 8);
                        double a0 = 0.0, b0 = 0.0;
                        for (int q = 0; q < c.stp; ++q) {
                            a0 += lds64(pr + 8 * q);
                            b0 += lds64(pr + 8 * q + (unsigned)(PF * kPartPitch * 8));
                        }
                        const unsigned ta = it.tab + (unsigned)((g * it.SL + (kwb + sl - kw_base)) * 8);
                        sts64(ta, a0);
                        sts64(ta + gofs, b0);
                    }
                    __syncwarp();
                }
            }
        }
        if (++bis == it.KB) {
            __syncwarp();
            score_narrow<DBG>(c, best, lane, it.G, it.SL, it.SLn, it.invSL, kw_base, it.L);
            __syncwarp();
            kw_base += it.SLn;
            bis = 0;
        }
    }
    cp_async_wait<0>();
    if (bis > 0) {
        __syncwarp();
        score_narrow<DBG>(c, best, lane, it.G, it.SL, it.SLn, it.invSL, kw_base, it.L);
        __syncwarp();
    }
}

// Wide path, one segment per warp, as a SHIFT REGISTER: acc[j] is the partial sum of the window that has
// taken j taps so far; a row step is  acc[j+1] = T[j] * x + acc[j]  for j = MB-1 .. 1 (the destination of a
// DFMA is not its addend, so nothing is moved), acc[1] = T[0] * x starts a window and acc[MB] is complete.
// All register indices are static after unrolling ONE batch of 8 rows (the ring form needed MB rows), so the
// body is 8 * MB DFMAs and the whole steady state is branch free:
//   - the X FIFO is three groups of 8 rows; when the reads (3 rows ahead of the multiplies) enter the next
//     group, the 8 slots just left are refilled by predicated zero-filling 8-byte cp.async copies, 19 - 26
//     rows ahead of their use;
//   - the column sums of batch b-1 (8 windows x 32 lanes in the emit buffer: four lanes per window, eight
//     strided values each, two shuffle steps, then table[row] += sum) are spread over rows 0 .. 4 of batch b;
//     the two emit buffers alternate.
// Table entry rho holds the window that COMPLETES at row rho of the tile, i.e. window rho - (MB-1): the
// first MB-1 entries (warm-up rows) and the 8 entries behind the table proper (the sums the first batch
// takes from the still empty emit buffer) are slack that is never scored, so no store is predicated.
constexpr int kSPF = 8;                         // rows per batch
constexpr int kTabSlack = 8;                    // dummy entries behind the rows of a table
constexpr int kChunkW = 31;                     // columns per chunk: any 31 consecutive doubles lie inside 16 aligned 16-byte pieces
// X feed: a cp.async instruction costs the issuing sub-partition ~11 cycles of FP64 issue whatever its size
// (measured: DFMA stream + one LDGSTS per k DFMAs), so the rows are copied in 16-byte pieces, TWO rows per
// instruction: lanes 0-15 copy the 16 pieces of one row (the aligned 32-double window around the chunk's
// 31 columns), lanes 16-31 the next row.  Lane l then reads its own column at (l + parity) * 8 of the row
// slot, parity = (first element of the row) & 1; rows alternate between two parities when stp is odd, and a
// lane half always copies rows of the same parity (its pointer advances by 2 stp per copy).
template <int MB, typename F>
__device__ __forceinline__ void march_shift(const Cls& c, const unsigned tab, const unsigned tab_dummy,
                                            const double* __restrict__ x, const long long ebase0,
                                            const int rows_valid, const int nbat, const F (&T)[MB],
                                            const int lane) {
    constexpr int PF = kSPF, XQ = 4, LA = 3, NG = 3;
    static_assert(NG * PF <= kFifoRows && 2 * PF <= kPartRows && MB >= 2, "geometry");
    constexpr unsigned kRowB = kPartPitch * 8;     // bytes per emit-buffer row
    constexpr unsigned kGrpB = PF * 256;           // bytes per FIFO group
    F acc[MB + 1], xq[XQ];
#pragma unroll
    for (int u = 0; u <= MB; ++u) acc[u] = (F)0;
    // copy role: rows 2j + half of a group, piece `pc` (two doubles) of the row's aligned window
    const int half = lane >> 4, pc = lane & 15;
    const double* cp = x + (((ebase0 + (long long)half * c.stp) >> 1) << 1) + 2 * pc;
    const long long cstride = 2ll * c.stp;
    const unsigned cdst = c.fifo + (unsigned)(half * 256 + pc * 16);
    int row_issue = half;                          // row index of this lane's next copy
#pragma unroll
    for (int k = 0; k < NG; ++k) {
#pragma unroll
        for (int j = 0; j < PF / 2; ++j) {
            cp_async16(cdst + (unsigned)((k * PF + 2 * j) * 256), cp, row_issue < rows_valid);
            cp += cstride;
            row_issue += 2;
        }
        cp_async_commit();
    }
    cp_async_wait<NG - 1>();
    __syncwarp();
    // read role: own column of even / odd rows of a batch (PF is even: the same parities in every batch)
    const int p0 = (int)(ebase0 & 1), p1 = (int)((ebase0 + c.stp) & 1);
    const unsigned fe = c.fifo + (unsigned)((lane + p0) * 8), fo = c.fifo + (unsigned)((lane + p1) * 8);
#pragma unroll
    for (int k = 0; k < LA; ++k) xq[k] = (F)lds64(((k & 1) ? fo : fe) + (unsigned)(k * 256));
    unsigned gcur = 0, gnext = kGrpB;              // byte offsets of the FIFO group being multiplied / the next

    // column-sum roles: lane = (window slot sl, quarter r); quarter r adds lanes r, r+4, ..., r+28
    const int sl = lane >> 2, r = lane & 3;
    const unsigned rd_off = (unsigned)((sl * kPartPitch + r) * 8);
    unsigned pcur = c.part + (unsigned)(lane * 8);            // emit buffer of the running batch (my column)
    unsigned pother = pcur + (unsigned)(PF * kRowB);
    unsigned rprev = c.part + (unsigned)(PF * kRowB) + rd_off;   // batch being summed (first: empty buffer -> dummy)
    unsigned tprev = tab_dummy + (unsigned)(sl * 8);
    double v0 = 0.0, v1 = 0.0, v2 = 0.0, v3 = 0.0, sa = 0.0, ta = 0.0;

#pragma unroll 1
    for (int b = 0; b < nbat; ++b) {
#pragma unroll
        for (int u = 0; u < PF; ++u) {
            if (u + LA == PF) {
                // the reads enter the next group: refill the group just read, make sure the next one landed
#pragma unroll
                for (int j = 0; j < PF / 2; ++j) {
                    cp_async16(cdst + gcur + (unsigned)(2 * j * 256), cp, row_issue < rows_valid);
                    cp += cstride;
                    row_issue += 2;
                }
                cp_async_commit();
                cp_async_wait<NG - 1>();
                __syncwarp();                      // the pieces of a row come from 16 lanes
            }
            {
                const int q = u + LA;              // row (of this batch) being read
                const unsigned fb = (q & 1) ? fo : fe;
                xq[q % XQ] = (F)lds64(q < PF ? fb + gcur + (unsigned)(q * 256) : fb + gnext + (unsigned)((q - PF) * 256));
            }
            const F xv = xq[u % XQ];
#pragma unroll
            for (int m = MB - 1; m >= 1; --m) acc[m + 1] = fma(T[m], xv, acc[m]);
            acc[1] = T[0] * xv;                                     // a window starts at this row
            sts64(pcur + (unsigned)(u * kRowB), (double)acc[MB]);   // the window that took its last tap
            // column sums of the previous batch, one stage per row
            if (u == 0) {
                sa = (v0 + v1) + (v2 + v3);
                v0 = lds64(rprev + 128); v1 = lds64(rprev + 160); v2 = lds64(rprev + 192); v3 = lds64(rprev + 224);
            } else if (u == 1) {
                sa += (v0 + v1) + (v2 + v3);
            } else if (u == 2) {
                sa += __shfl_xor_sync(0xffffffffu, sa, 1);
            } else if (u == 3) {
                sa += __shfl_xor_sync(0xffffffffu, sa, 2);
                ta = lds64(tprev);
            } else if (u == 4) {
                sts64(tprev, ta + sa);         // the four lanes of a slot store the same value
            }
        }
        __syncwarp();                              // this batch's emit rows are complete
        rprev = (pcur - (unsigned)(lane * 8)) + rd_off;
        tprev = tab + (unsigned)((b * PF + sl) * 8);
        v0 = lds64(rprev); v1 = lds64(rprev + 32); v2 = lds64(rprev + 64); v3 = lds64(rprev + 96);
        { const unsigned tmp = pcur; pcur = pother; pother = tmp; }
        gcur = gnext;
        gnext = gnext + kGrpB == NG * kGrpB ? 0u : gnext + kGrpB;
    }
    // drain: the last batch's sums
    sa = (v0 + v1) + (v2 + v3);
    v0 = lds64(rprev + 128); v1 = lds64(rprev + 160); v2 = lds64(rprev + 192); v3 = lds64(rprev + 224);
    sa += (v0 + v1) + (v2 + v3);
    sa += __shfl_xor_sync(0xffffffffu, sa, 1);
    sa += __shfl_xor_sync(0xffffffffu, sa, 2);
    sts64(tprev, lds64(tprev) + sa);
    cp_async_wait<0>();
    __syncwarp();
}

__device__ __forceinline__ double tmpl_lerp(const double* __restrict__ tm, int n_tmpl, int j, double tscale) {
    const double u = ((double)j + 0.5) * tscale;
    int k = (int)u;                                   // u >= 0: truncation == floor
    k = k > n_tmpl - 2 ? n_tmpl - 2 : k;
    const double fr = u - (double)k;
    const double t0 = tm[k];
    return t0 + fr * (tm[k + 1] - t0);
}

// One march of the lanes' (segment, column) slots: taps, bounds, then the ring.
//   seg/col: this lane's slot (active == false: an idle lane, zero taps);  row0: first row of seg.
template <int MB, bool NARROW, typename F, bool DUAL = false, bool DBG = false>
__device__ __forceinline__ void run_march(const Cls& c, const It& it, const int n, const int n_tmpl,
                                          const double tscale, const double* __restrict__ tm,
                                          const double* __restrict__ x, const bool square,
                                          const bool active, const int row0, const int col,
                                          const int lane, Cand& best,
                                          const double* __restrict__ xw = nullptr) {
    F T[MB];                                                         // taps: fp64 template, rounded once to F
#pragma unroll
    for (int m = 0; m < MB; ++m) {
        const int j = m * c.stp + col;
        double g = 0.0;
        if (active && j < c.D) g = tmpl_lerp(tm, n_tmpl, j, tscale);
        T[m] = (F)(square ? g * g : g);
    }
    const int nblk = (it.L + MB - 1 + MB - 1) / MB;
    const int rows_all = nblk * MB + kFifoBatches * PfRows<MB>::v;   // rows ever requested
    const long long lim = (long long)n + c.D;                        // x entries >= lim are never needed
    const long long ebase = (long long)c.off + (long long)row0 * c.stp + col;
    int rows_valid = 0;
    if (ebase < lim) {
        const long long rv = (lim - ebase + c.stp - 1) / c.stp;
        rows_valid = rv > rows_all ? rows_all : (int)rv;
    }
    const int rows_min = __reduce_min_sync(0xffffffffu, rows_valid);
    if constexpr (DUAL) march_dual<MB, F, DBG>(c, it, x + ebase, xw + ebase, rows_valid, rows_min, nblk, T, lane, best);
    else march<MB, NARROW, F, DBG>(c, it, x + ebase, rows_valid, rows_min, nblk, T, lane, best);
}

template <int MB, bool NARROW, bool UNIFORM, typename F, bool DBG = false>
__device__ __forceinline__ void run_class(const Cls& c, const int n, const int n_tmpl, const double tscale,
                                          const double* __restrict__ tm, const double* __restrict__ x1,
                                          const double* __restrict__ x0, const int lane, Cand& best) {
    if (c.nWr <= 0) return;
    if constexpr (NARROW) {
        It it;
        it.tab = c.ctab;
        // ---- narrow: G segments side by side, one march over the whole class -------------------
        it.direct = c.stp == 1;   // (stp <= kChi2NarrowMax; dy not uniform: C and G in one march, rings <= 16)
        it.G = 32 / c.stp;
        it.L = (c.nWr + it.G - 1) / it.G;
        it.KB = c.Kt / (it.G * MB);
        if (it.G * ((it.KB * MB) | 1) > c.Kt) --it.KB;       // odd pitch must still fit (KB >= 1 always)
        it.SLn = it.KB * MB;
        it.SL = it.SLn | 1;
        it.invSL = 1.0f / (float)it.SL;
        it.nWt = c.nWr;
        const bool active = lane < it.G * c.stp;
        const int seg = min(lane / c.stp, it.G - 1);
        const int col = lane - seg * c.stp;      // idle lanes read on behind the last segment (zero taps)
        if constexpr (UNIFORM)
            run_march<MB, true, F, false, DBG>(c, it, n, n_tmpl, tscale, tm, x1, false, active, seg * it.L, col, lane, best);
        else
            run_march<MB, true, F, true, DBG>(c, it, n, n_tmpl, tscale, tm, x1, false, active, seg * it.L, col, lane, best, x0);
    } else {
    // ---- wide: window tiles of the table size; the tile's stp columns are cut into nc balanced chunks of
    // at most 32 lanes, one shift march per chunk over all rows of the tile (one segment per warp: a few idle
    // lanes when stp is just above a multiple of 32, but no halo rows between segments).  c.Kt = table
    // entries per quantity: rows of the tile + kTabSlack dummy entries.
    const int Lmax = c.Kt - kTabSlack - (MB - 1);        // windows per tile (Kt - kTabSlack is a multiple of 8)
    const unsigned dummy = (unsigned)((c.Kt - kTabSlack) * 8);
    const int nc = (c.stp + kChunkW - 1) / kChunkW;
    const int cw = (c.stp + nc - 1) / nc;                // balanced chunks of at most 31 columns
    const long long lim = (long long)n + c.D;            // x entries >= lim are never needed
    for (int k0 = 0; k0 < c.nWr; k0 += Lmax) {
        const int nWt = min(Lmax, c.nWr - k0);
        const int nbat = (nWt + MB - 1 + kSPF - 1) / kSPF;
        const int rows_all = nbat * kSPF + 3 * kSPF;     // rows ever requested by a march
        for (int i = lane; i < nbat * kSPF; i += 32) {
            sts64(c.ctab + (unsigned)(i * 8), 0.0);
            if (!c.uniform) sts64(c.ctab + (unsigned)((c.Kt + i) * 8), 0.0);
        }
        __syncwarp();
        for (int pass = 0; pass < (c.uniform ? 1 : 2); ++pass) {
            const unsigned tab = c.ctab + (unsigned)(pass * c.Kt * 8);
            const double* __restrict__ x = pass == 0 ? x1 : x0;
            for (int ch = 0; ch < nc; ++ch) {
                const int col = ch * cw + lane;          // idle lanes (zero taps) read what the row copies bring
                const bool active = lane < cw && col < c.stp;
                F T[MB];                                 // taps: fp64 template, rounded once to F
#pragma unroll
                for (int m = 0; m < MB; ++m) {
                    const int j = m * c.stp + col;
                    double g = 0.0;
                    if (active && j < c.D) g = tmpl_lerp(tm, n_tmpl, j, tscale);
                    T[m] = (F)(pass == 1 ? g * g : g);
                }
                // rows whose first element is < lim are copied (32 doubles from the aligned start: they stay
                // inside the period's pad + zero margin, k_durtab); later rows are zero-filled
                const long long ebase0 = (long long)c.off + (long long)k0 * c.stp + ch * cw;
                int rows_valid = 0;
                if (ebase0 < lim) {
                    const long long rv = (lim - ebase0 + c.stp - 1) / c.stp;
                    rows_valid = rv > rows_all ? rows_all : (int)rv;
                }
                march_shift<MB, F>(c, tab, tab + dummy, x, ebase0, rows_valid, nbat, T, lane);
            }
        }
        __syncwarp();
        score_wide<DBG>(c, best, lane, k0, nWt, MB - 1);
        __syncwarp();
    }
    }
}

template <int MB, bool NARROW, bool UNIFORM, typename F, bool DBG = false>
__global__ void __launch_bounds__(kRT, 6) k_chi2_ring(TileArgs a, const int* __restrict__ list,
                                                      const int* __restrict__ count, int* __restrict__ next) {
    extern __shared__ double dsm[];                 // per warp: emit buffer, X FIFO, window table
    __shared__ __align__(16) double s_tmpl[kTmplSmem];
    __shared__ __align__(8) unsigned long long s_mbar;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n_mine = *count;                      // trials of this variant in the tile
    if ((int)blockIdx.x * kRW >= n_mine) return;    // (more CTAs than trials)
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
    // ---- from here on every warp works alone: it takes the next trial of the variant's list from a
    // device-wide counter (persistent CTAs, one wave: a warp is idle only when the list is empty) --------
    for (;;) {
    int li = 0;
    if (lane == 0) li = atomicAdd(next, 1);
    li = __shfl_sync(0xffffffffu, li, 0);
    if (li >= n_mine) break;
    const int trial = list[li];
    const int pl = trial / a.n_dur;
    const DurEntry e = a.durtab[trial];
    Partial* out = a.partial + trial;
    const int st = e.stride;
    const int nW = (a.n + st - 1) / st;
    const int M = (e.D + st - 1) / st;
    const int ncls = chi2_classes(M, st, UNIFORM);           // window classes: at most MB taps each
    Cls c;
    c.D = e.D; c.stp = ncls * st;
    c.uniform = UNIFORM;
    c.gbar = e.gbar;
    c.G_u = a.w_uniform * e.gg2;
    c.inv_den_u = __ddiv_rn(1.0, ((double)e.D * a.w_uniform) * e.gbar);
    c.s1 = a.s1 + (long long)pl * a.spitch;
    c.s0 = a.s0 + (long long)pl * a.spitch;
    double* const wsm = dsm + warp * WarpSmem<NARROW>::v;
    c.part = (unsigned)__cvta_generic_to_shared(wsm);
    c.fifo = c.part + (unsigned)(kPartRows * kPartPitch * 8);
    c.ctab = c.fifo + (unsigned)(kFifoRows * 32 * 8);
    c.Kt = NARROW ? (UNIFORM ? kCW : kCW / 2) : (UNIFORM ? kCWWide : kCWWide / 2);
    c.dbg_d = a.dbg_dchi2; c.dbg_a = a.dbg_depth; c.st0 = st;
    const double tscale = __ddiv_rn((double)(a.n_tmpl - 1), (double)e.D);
    const double* __restrict__ tm = tmpl_in_smem ? s_tmpl : a.tmpl;
    const double* __restrict__ x1 = a.x1 + (long long)pl * a.pitch;
    const double* __restrict__ x0 = a.x0 + (long long)pl * a.pitch;
    Cand best; best.has = 0; best.d = 0.0; best.s = 0; best.depth = 0.0;

    for (int r = 0; r < ncls; ++r) {
        c.off = r * st;
        c.nWr = nW > r ? (nW - r + ncls - 1) / ncls : 0;
        run_class<MB, NARROW, UNIFORM, F, DBG>(c, a.n, a.n_tmpl, tscale, tm, x1, x0, lane, best);
    }

    // warp-wide lexicographic min on (d, s)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        Cand o2;
        o2.d = __shfl_xor_sync(0xffffffffu, best.d, o);
        o2.depth = __shfl_xor_sync(0xffffffffu, best.depth, o);
        o2.s = __shfl_xor_sync(0xffffffffu, best.s, o);
        o2.has = __shfl_xor_sync(0xffffffffu, best.has, o);
        if (o2.has) cand_offer(best, o2.d, o2.s, o2.depth);
    }
    if (lane == 0) { out->valid = best.has; out->dchi2 = best.d; out->depth = best.depth; out->start = best.s; }
    __syncwarp();
    }
}

}  // namespace

template <int MB, bool NARROW, bool UNIFORM, typename F>
static void launch_variant_t(const TileArgs& a, int v, cudaStream_t st) {
    const long long trials = (long long)a.tile * a.n_dur;
    unsigned grid = (unsigned)((trials + kRW - 1) / kRW);           // surplus CTAs exit at once
    if (grid > kGridCap) grid = kGridCap;                           // one wave of persistent CTAs
    // wide variants: 3 CTAs per SM (their 60 KB of shared memory each: kCWWide).  The shift march hides its latencies
    // inside a warp (6 - 8 warps per SM run within 1 % of 12), and fewer trials in flight are fewer periods whose x1 competes for the L2
    // (c4: 60 -> 36 GB of DRAM reads per 4144-period tile of the dominant variant, SM clock under the power cap 1845 -> 1890 MHz)
    if (!NARROW && grid > kGridCapWide) grid = kGridCapWide;
    const size_t sm = (size_t)(kRW * WarpSmem<NARROW>::v) * sizeof(double);
    // (per device, cheap: set on every launch rather than behind a process-wide flag)
    cudaFuncSetAttribute(k_chi2_ring<MB, NARROW, UNIFORM, F>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if constexpr (sizeof(F) == 8) {
        if (a.dbg_dchi2) {       // gtls_ring_window_chi2: the same kernel, instantiated to dump every window's score
            cudaFuncSetAttribute(k_chi2_ring<MB, NARROW, UNIFORM, F, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
            k_chi2_ring<MB, NARROW, UNIFORM, F, true><<<grid, kRT, sm, st>>>(a, a.trial_list + (long long)v * trials, a.trial_count + v,
                                                                           a.trial_count + kChi2Variants * (1 + kBinBlocks) + v);
            return;
        }
    }
    k_chi2_ring<MB, NARROW, UNIFORM, F><<<grid, kRT, sm, st>>>(a, a.trial_list + (long long)v * trials, a.trial_count + v,
                                                             a.trial_count + kChi2Variants * (1 + kBinBlocks) + v);
}
// fp64 ring (default) or the fp32 in-transit variant (gtls_opts.chi2_fp32: taps, X and the ring
// accumulators in fp32 -- at most 24 products per sum; column sums, prefix sums and scoring stay fp64)
template <int MB, bool NARROW, bool UNIFORM>
static void launch_variant(const TileArgs& a, int v, cudaStream_t st) {
    if (a.chi2_fp32) launch_variant_t<MB, NARROW, UNIFORM, float>(a, v, st);
    else launch_variant_t<MB, NARROW, UNIFORM, double>(a, v, st);
}

void launch_chi2_ring(const TileArgs& a, cudaStream_t st) {
    launch_bin_trials(a, st);
    cudaStream_t ss = st;
    SideStream* side = side_stream(0);
    if (side) {
        cudaEventRecord(side->fork, st);
        cudaStreamWaitEvent(side->s, side->fork, 0);
        ss = side->s;
    }
    if (a.uniform) {
        launch_variant<12, true, true>(a, 9, ss);
        launch_variant<16, true, true>(a, 8, ss);
        launch_variant<8, true, true>(a, 10, ss);
        launch_variant<4, true, true>(a, 11, ss);
        launch_variant<24, true, true>(a, 6, ss);
        launch_variant<21, true, true>(a, 7, ss);
        launch_variant<16, false, true>(a, 2, ss);
        launch_variant<12, false, true>(a, 3, ss);
        launch_variant<8, false, true>(a, 4, ss);
        launch_variant<4, false, true>(a, 5, ss);
        launch_variant<21, false, true>(a, 1, st);
    } else {
        launch_variant<12, true, false>(a, 9, ss);
        launch_variant<16, true, false>(a, 8, ss);
        launch_variant<8, true, false>(a, 10, ss);
        launch_variant<4, true, false>(a, 11, ss);
        launch_variant<16, false, false>(a, 2, ss);
        launch_variant<12, false, false>(a, 3, ss);
        launch_variant<8, false, false>(a, 4, ss);
        launch_variant<4, false, false>(a, 5, ss);
        launch_variant<21, false, false>(a, 1, st);
    }
    if (side) {
        cudaEventRecord(side->join, ss);
        cudaStreamWaitEvent(st, side->join, 0);
    }
}

}  // namespace gtls
