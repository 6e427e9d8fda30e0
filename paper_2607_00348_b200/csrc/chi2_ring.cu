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
constexpr int kCW = 704;                 // window-table doubles per warp (>= 32 * 21)
constexpr int kTmplSmem = 512;           // template nodes cached in shared memory
#ifndef GTLS_GRID_WAVES
#define GTLS_GRID_WAVES 16
#endif
constexpr unsigned kGridCap = 148u * 6u * GTLS_GRID_WAVES;   // CTAs per launch: waves of the 6 resident CTAs per SM
// The cap applies to short light curves only: there the trials are short and tens of thousands of empty CTAs
// per variant launch are 5 % of a search (c2 9.73 -> 9.14 ms, c1 1.70 -> 1.63 ms; 8 / 16 / 32 waves: c2 9.27 / 9.14 / 9.15 ms).  On long curves the fixed
// round-robin assignment of trials to warps loses more at the tail than the empty CTAs cost (c4 6.2 -> 6.7 s,
// c3 1.54 -> 1.70 s with the cap): there every CTA takes one pair of trials and the hardware balances them.
constexpr int kGridCapMaxN = 16384;
constexpr int kWarpSmem = kPartRows * kPartPitch + kFifoRows * 32 + kCW;   // doubles per warp

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
};

// a5 + a8 for one window kappa of the class (start s = off + kappa*stp): hi/lo are the prefix sums
// at s+D and s.  a = max(rbar, 0) / mean(g_D) with rbar = swr / sw.  Uniform dy: sw * mean(g_D) is a
// constant of the trial, so a = max(swr, 0) * inv_den (one multiply); otherwise one division.
__device__ __forceinline__ void score_one(const Cls& c, Cand& best, const int s, const double hi1,
                                          const double lo1, const double hi0, const double lo0,
                                          const double C, const double Gt) {
    const double swr = fmax(hi1 - lo1, 0.0);
    const double depth = c.uniform ? swr * c.inv_den_u : __ddiv_rn(swr, (hi0 - lo0) * c.gbar);
    const double Gv = c.uniform ? c.G_u : Gt;
    const double d = -2.0 * depth * C + (depth * depth) * Gv;
    if (d <= best.d || !best.has) cand_offer(best, d, s, depth);     // rarely taken after the first windows
}
// Wide path: score the windows [k0, k0 + nWt) of the class from table entries [0, nWt).
__device__ __forceinline__ void score_wide(const Cls& c, Cand& best, const int lane, const int k0,
                                           const int nWt) {
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
                const unsigned ta = c.ctab + (unsigned)(w * 8);
                score_one(c, best, c.off + (k0 + w) * c.stp, hi1[u], lo1[u], hi0[u], lo0[u], lds64(ta),
                          c.uniform ? 0.0 : lds64(ta + (unsigned)(c.Kt * 8)));
            }
        }
    }
}

// Narrow path: table entry seg*SL + o holds window kw = kw_base + o of segment seg (kappa = seg*L + kw).
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
                score_one(c, best, sidx[u], hi1[u], lo1[u], hi0[u], lo0[u], lds64(ta),
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
template <int MB, bool NARROW, typename F>
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
            score_narrow(c, best, lane, it.G, it.SL, it.SLn, it.invSL, kw_base, it.L);
            __syncwarp();
            kw_base += it.SLn;
            bis = 0;
        }
    }
    cp_async_wait<0>();
    if (NARROW && bis > 0) {
        __syncwarp();
        score_narrow(c, best, lane, it.G, it.SL, it.SLn, it.invSL, kw_base, it.L);
        __syncwarp();
    }
}

// Narrow path when dy is NOT uniform: C = sum g x1 and G = sum g^2 x0 are needed for every window of the
// time-sliced table, so both are accumulated in ONE march: two rings (C, G) over two FIFO streams
// (x1 = w r, x0 = w), taps g held once (g^2 x0 is taken as g * (g * x0)).  3 MB doubles of ring state:
// ring sizes up to 16.  Batches of kDualPF rows per stream, the two streams share the FIFO half and half;
// the emit buffer holds the C partials in rows [0, PF) and the G partials in rows [PF, 2 PF).
constexpr int kDualPF = 4;
template <int MB, typename F>
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
            score_narrow(c, best, lane, it.G, it.SL, it.SLn, it.invSL, kw_base, it.L);
            __syncwarp();
            kw_base += it.SLn;
            bis = 0;
        }
    }
    cp_async_wait<0>();
    if (bis > 0) {
        __syncwarp();
        score_narrow(c, best, lane, it.G, it.SL, it.SLn, it.invSL, kw_base, it.L);
        __syncwarp();
    }
}

// Wide path, one segment per warp: the same march as a software pipeline.  A warp issues in order, so
// every load is placed at least one row (MB DFMAs) before its first use:
//   - the X value of row j+LA is read from the FIFO while row j is multiplied; whenever the reads enter a
//     new group of PF rows, the PF slots of the group just left are refilled (cp.async) with their rows
//     + MB in one burst (FIFO depth = MB rows);
//   - the column sums of a completed batch of PF windows are spread over the rows of the NEXT batch:
//     A (batch end) 4 loads, B 4 loads + first partial sum, C second partial sum, D/E the two shuffle
//     steps and the table load, F the table store.  Two emit buffers alternate.
template <int MB, typename F>
__device__ __forceinline__ void march_pipe(const Cls& c, const It& it, const double* __restrict__ xp,
                                           const int rows_valid, const int rows_min, const int nblk,
                                           const F (&T)[MB], const int lane) {
    constexpr int PF = PfRows<MB>::v;
    constexpr int NBAT = MB / PF;                  // copy groups in flight = batches per block
    constexpr int XQ = (MB % 3 == 0) ? 3 : 4;      // X registers; LA rows of look-ahead
    constexpr int LA = XQ - 1;
    static_assert(PF >= 6 && MB % PF == 0 && MB % XQ == 0 && MB <= kFifoRows && 2 * PF <= kPartRows, "geometry");
    constexpr unsigned kRowB = kPartPitch * 8;     // bytes per emit-buffer row
    F acc[MB], xq[XQ];
#pragma unroll
    for (int u = 0; u < MB; ++u) acc[u] = (F)0;
    const unsigned fl = c.fifo + (unsigned)(lane * 8);
    const long long rstride = (long long)c.stp;
    int row_issue = 0;                             // next row to copy
#pragma unroll
    for (int k = 0; k < NBAT; ++k) {
#pragma unroll
        for (int u = 0; u < PF; ++u) {
            cp_async8(fl + (unsigned)((k * PF + u) * 256), xp, row_issue < rows_valid);
            xp += rstride;
            ++row_issue;
        }
        cp_async_commit();
    }
    cp_async_wait<NBAT - 1>();
#pragma unroll
    for (int k = 0; k < LA; ++k) xq[k] = (F)lds64(fl + (unsigned)(k * 256));

    // column-sum roles: lane = (window slot sl, quarter r); quarter r adds lanes r, r+4, ..., r+28
    const int sl = lane >> 2, r = lane & 3;
    const int slc = sl < PF ? sl : PF - 1;
    const unsigned rd_off = (unsigned)((slc * kPartPitch + r) * 8);
    const bool my_slot = r == 0 && sl < PF;
    const unsigned tab0 = it.tab + (unsigned)(sl * 8);
    unsigned pcur = c.part + (unsigned)(lane * 8);            // emit buffer of the running batch (my column)
    unsigned pother = pcur + (unsigned)(PF * kRowB);
    unsigned rprev = c.part + rd_off;                         // read base of the batch being summed
    int kw_prev = -(1 << 30);                                 // no previous batch yet
    double v0 = 0.0, v1 = 0.0, v2 = 0.0, v3 = 0.0, sa = 0.0, ta = 0.0;
    bool oka = false;

#pragma unroll 1
    for (int blk = 0; blk < nblk; ++blk) {
#pragma unroll
        for (int u = 0; u < MB; ++u) {
            if ((u + LA) % PF == 0) {
                // the reads enter a new group: refill the group just left, then make sure the new one landed
                const int g0 = ((u + LA - PF) % MB + MB) % MB;   // (compile-time after unrolling)
                if (row_issue + PF <= rows_min) {
#pragma unroll
                    for (int k = 0; k < PF; ++k) { cp_async8(fl + (unsigned)((g0 + k) * 256), xp); xp += rstride; }
                } else {
#pragma unroll
                    for (int k = 0; k < PF; ++k) { cp_async8(fl + (unsigned)((g0 + k) * 256), xp, row_issue + k < rows_valid); xp += rstride; }
                }
                row_issue += PF;
                cp_async_commit();
                cp_async_wait<NBAT - 1>();
            }
            xq[(u + LA) % XQ] = (F)lds64(fl + (unsigned)(((u + LA) % MB) * 256));
            const F x = xq[u % XQ];
#pragma unroll
            for (int m = 0; m < MB; ++m) {
                const int a = (u - m + MB) % MB;
                if (m == 0) acc[a] = T[0] * x;                      // window gamma starts at this row
                else acc[a] = fma(T[m], x, acc[a]);
            }
            sts64(pcur + (unsigned)((u % PF) * kRowB), (double)acc[(u + 1) % MB]);   // window gamma-(MB-1) complete
            // column sums of the previous batch, one stage per row
            if (u % PF == 0) {
                sa = (v0 + v1) + (v2 + v3);
                v0 = lds64(rprev + 128); v1 = lds64(rprev + 160); v2 = lds64(rprev + 192); v3 = lds64(rprev + 224);
            } else if (u % PF == 1) {
                sa += (v0 + v1) + (v2 + v3);
            } else if (u % PF == 2) {
                sa += __shfl_xor_sync(0xffffffffu, sa, 1);
            } else if (u % PF == 3) {
                sa += __shfl_xor_sync(0xffffffffu, sa, 2);
                const int kw = kw_prev + sl;
                oka = my_slot && kw >= 0 && kw < it.L && kw < it.nWt;
                ta = oka ? lds64(tab0 + (unsigned)(kw_prev * 8)) : 0.0;
            } else if (u % PF == 4) {
                if (oka) sts64(tab0 + (unsigned)(kw_prev * 8), ta + sa);
            }
            if (u % PF == PF - 1) {                                 // batch complete: it becomes "previous"
                __syncwarp();
                rprev = (pcur - (unsigned)(lane * 8)) + rd_off;
                v0 = lds64(rprev); v1 = lds64(rprev + 32); v2 = lds64(rprev + 64); v3 = lds64(rprev + 96);
                kw_prev = blk * MB + (u - (PF - 1)) - (MB - 1);
                const unsigned tmp = pcur; pcur = pother; pother = tmp;
            }
        }
    }
    // drain: the last batch's sums
    sa = (v0 + v1) + (v2 + v3);
    v0 = lds64(rprev + 128); v1 = lds64(rprev + 160); v2 = lds64(rprev + 192); v3 = lds64(rprev + 224);
    sa += (v0 + v1) + (v2 + v3);
    sa += __shfl_xor_sync(0xffffffffu, sa, 1);
    sa += __shfl_xor_sync(0xffffffffu, sa, 2);
    {
        const int kw = kw_prev + sl;
        if (my_slot && kw >= 0 && kw < it.L && kw < it.nWt)
            tab_add(tab0 + (unsigned)(kw_prev * 8), sa);
    }
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
template <int MB, bool PIPE, bool NARROW, typename F, bool DUAL = false>
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
    if constexpr (DUAL) march_dual<MB, F>(c, it, x + ebase, xw + ebase, rows_valid, rows_min, nblk, T, lane, best);
    else if constexpr (PIPE) march_pipe<MB, F>(c, it, x + ebase, rows_valid, rows_min, nblk, T, lane);
    else march<MB, NARROW, F>(c, it, x + ebase, rows_valid, rows_min, nblk, T, lane, best);
}

template <int MB, bool NARROW, bool UNIFORM, typename F>
__device__ __forceinline__ void run_class(const Cls& c, const int n, const int n_tmpl, const double tscale,
                                          const double* __restrict__ tm, const double* __restrict__ x1,
                                          const double* __restrict__ x0, const int lane, Cand& best) {
    if (c.nWr <= 0) return;
    It it;
    it.tab = c.ctab;
    if constexpr (NARROW) {
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
            run_march<MB, false, true, F>(c, it, n, n_tmpl, tscale, tm, x1, false, active, seg * it.L, col, lane, best);
        else
            run_march<MB, false, true, F, true>(c, it, n, n_tmpl, tscale, tm, x1, false, active, seg * it.L, col, lane, best, x0);
        return;
    }
    // ---- wide: window tiles of the table size; the tile's stp columns are cut into nc balanced chunks of
    // at most 32 lanes, one march per chunk over all rows of the tile (one segment per warp: a few idle
    // lanes when stp is just above a multiple of 32, but no halo rows between segments and every march
    // takes the pipelined path).
    it.direct = false;
    it.G = 0; it.KB = 0; it.SL = 0; it.SLn = 0; it.invSL = 0.f;
    constexpr bool kPipe = PfRows<MB>::v >= 6;
    const int nc = (c.stp + 31) >> 5;
    const int cw = (c.stp + nc - 1) / nc;
    for (int k0 = 0; k0 < c.nWr; k0 += c.Kt) {
        const int nWt = min(c.Kt, c.nWr - k0);
        it.L = nWt;
        it.nWt = nWt;
        for (int i = lane; i < (c.uniform ? nWt : c.Kt + nWt); i += 32) sts64(c.ctab + (unsigned)(i * 8), 0.0);
        __syncwarp();
        for (int pass = 0; pass < (c.uniform ? 1 : 2); ++pass) {
            it.tab = c.ctab + (unsigned)(pass * c.Kt * 8);
            for (int ch = 0; ch < nc; ++ch) {
                const int c0 = ch * cw;
                const bool active = lane < cw && c0 + lane < c.stp;
                const int col = c0 + lane;     // idle lanes read on behind the chunk (zero taps): the warp's
                                               // copies stay one contiguous, conflict-free 256-byte row
                run_march<MB, kPipe, false, F>(c, it, n, n_tmpl, tscale, tm, pass == 0 ? x1 : x0, pass == 1, active, k0,
                                     col, lane, best);
            }
        }
        __syncwarp();
        score_wide(c, best, lane, k0, nWt);
        __syncwarp();
    }
}

template <int MB, bool NARROW, bool UNIFORM, typename F>
__global__ void __launch_bounds__(kRT, 6) k_chi2_ring(TileArgs a, const int* __restrict__ list,
                                                      const int* __restrict__ count) {
    extern __shared__ double dsm[];                 // per warp: emit buffer, X FIFO, window table
    __shared__ __align__(16) double s_tmpl[kTmplSmem];
    __shared__ __align__(8) unsigned long long s_mbar;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n_mine = *count;                      // trials of this variant in the tile
    if ((int)blockIdx.x * kRW >= n_mine) return;
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
    // (grid-stride over the variant's trial list: for short light curves the grid is capped at GTLS_GRID_WAVES
    // waves of resident CTAs, see kGridCapMaxN; otherwise the loop runs once)
    for (int li = (int)blockIdx.x * kRW + warp; li < n_mine; li += (int)gridDim.x * kRW) {
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
    double* const wsm = dsm + warp * kWarpSmem;
    c.part = (unsigned)__cvta_generic_to_shared(wsm);
    c.fifo = c.part + (unsigned)(kPartRows * kPartPitch * 8);
    c.ctab = c.fifo + (unsigned)(kFifoRows * 32 * 8);
    c.Kt = UNIFORM ? kCW : kCW / 2;
    const double tscale = __ddiv_rn((double)(a.n_tmpl - 1), (double)e.D);
    const double* __restrict__ tm = tmpl_in_smem ? s_tmpl : a.tmpl;
    const double* __restrict__ x1 = a.x1 + (long long)pl * a.pitch;
    const double* __restrict__ x0 = a.x0 + (long long)pl * a.pitch;
    Cand best; best.has = 0; best.d = 0.0; best.s = 0; best.depth = 0.0;

    for (int r = 0; r < ncls; ++r) {
        c.off = r * st;
        c.nWr = nW > r ? (nW - r + ncls - 1) / ncls : 0;
        run_class<MB, NARROW, UNIFORM, F>(c, a.n, a.n_tmpl, tscale, tm, x1, x0, lane, best);
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
    unsigned grid = (unsigned)((trials + kRW - 1) / kRW);           // worst case; surplus CTAs exit at once
    if (a.n <= kGridCapMaxN && grid > kGridCap) grid = kGridCap;
    const size_t sm = (size_t)(kRW * kWarpSmem) * sizeof(double);
    static bool set = false;
    if (!set) {
        cudaFuncSetAttribute(k_chi2_ring<MB, NARROW, UNIFORM, F>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
        set = true;
    }
    k_chi2_ring<MB, NARROW, UNIFORM, F><<<grid, kRT, sm, st>>>(a, a.trial_list + (long long)v * trials, a.trial_count + v);
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
