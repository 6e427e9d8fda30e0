// Steps a5-a8, register-tiled in-transit chi2 ("rows" formulation) -- the dominant kernel.
//
// For one (period, duration) with D points per window and stride st between trial starts
// (Eq. 18), split the template index j = m*st + i (row m, column i < st).  Window k then reads
//     C[k] = sum_m sum_i g[m*st+i] * X[k+m][i],      X[rho][i] = x1[rho*st + i]
// i.e. the folded curve viewed as rows of st points, and window k covers rows k..k+M-1
// (M = ceil(D/st), ~20 for dt0 = 0.05).  A thread owns A = 15 consecutive windows and ONE
// column i; walking the A+MB-1 rows those windows touch it loads each X value once and uses
// it for up to A FMAs against MB template values held in registers:
//     (A + 2 MB - 1) shared-memory loads for A*MB FMAs  (56 loads : 315 DFMA for MB = 21),
// which keeps the fp64 FMA pipe (64/clk/SM), not shared memory (16 doubles/clk/SM), the limiter.
// Lanes of a warp cover a chunk of cw <= 32 columns (times G window groups when st is small),
// so X tiles are read conflict-free; the per-column partial sums are combined with a
// segmented shuffle reduction once per row tile.
//
// X tiles ([rows][cols] sub-blocks of x1, row pitch st in global memory, 8-byte aligned only)
// are staged with 8-byte cp.async (LDGSTS, zero-fill outside the curve) into a double buffer;
// the template is resampled (lerp at cell centres, G14) straight into shared memory per stage.
// With non-uniform dy a second pass accumulates G = sum g^2 x0 the same way.
#include "gtls_internal.cuh"

namespace gtls {

namespace {

constexpr int kA = 15;                    // windows per thread
constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;
constexpr int kSmemDoubles = 12800;       // 102.4 KB dynamic + 8 KB template -> 2 CTAs per SM
constexpr int kTmplSmem = 1024;           // template nodes cached in shared memory
constexpr int kMaxColsT = 64;             // columns staged per stage (WC * cw)

struct Geom {
    int D, st, nW, M, MB, nmb;
    int cw, nc;          // column chunk width, number of chunks (cw * nc >= st)
    int G;               // window groups per warp (lanes = G * cw <= 32)
    int WR, WC;          // warp grid: row-warps x column-warps (WR * WC <= 8)
    int RT;              // windows per row tile = WR * G * kA
    int rows;            // X rows per stage = RT + MB - 1
    int colsT;           // columns per stage = WC * cw
    int pitch;           // shared-memory row pitch of the X tile (doubles)
    int nrt, nccs, npass;
    int xs_off[2], gs_off[2], tot_off;   // offsets (doubles) into dynamic shared memory
    double tscale;       // (n_tmpl - 1) / D
};

struct Cand { double d; double depth; int s; int has; };

__device__ __forceinline__ void cand_offer(Cand& b, double d, int s, double depth) {
    if (!b.has || d < b.d || (d == b.d && s < b.s)) { b.d = d; b.s = s; b.depth = depth; b.has = 1; }
}

__device__ __forceinline__ void cp_async8(unsigned d, const double* src, bool valid) {
    const int sz = valid ? 8 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(d), "l"(src), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

// bank-conflict test for one candidate pitch: lanes (g, c) of each half-warp must hit distinct
// 8-byte bank pairs when reading X[(g*kA + gamma) * pitch + c].
__device__ bool pitch_ok(int pitch, int G, int cw) {
    for (int h = 0; h < 2; ++h) {
        unsigned mask = 0;
        for (int l = 16 * h; l < 16 * h + 16; ++l) {
            if (l >= G * cw) break;
            const int g = l / cw, c = l - g * cw;
            const unsigned bit = 1u << ((g * kA * pitch + c) & 15);
            if (mask & bit) return false;
            mask |= bit;
        }
    }
    return true;
}

__device__ void make_geom(Geom& q, int n, int D, int st, int n_tmpl, bool uniform) {
    q.D = D; q.st = st;
    q.nW = (n + st - 1) / st;
    q.M = (D + st - 1) / st;
    q.MB = q.M <= 7 ? 7 : (q.M <= 14 ? 14 : 21);
    q.nmb = (q.M + q.MB - 1) / q.MB;
    q.npass = uniform ? 1 : 2;
    q.tscale = __ddiv_rn((double)(n_tmpl - 1), (double)D);
    const int ngr = (q.nW + kA - 1) / kA;
    // column chunking: maximise (useful columns / staged columns) * (active lanes / 32)
    const int nc0 = (st + 31) / 32;
    int best_nc = nc0; float best_eff = -1.f;
    for (int nc = nc0; nc <= nc0 + 6 && nc <= st; ++nc) {
        const int cw = (st + nc - 1) / nc;
        int G = 32 / cw; if (G > ngr) G = ngr;
        const float eff = (float)st / (float)(nc * cw) * (float)(G * cw) / 32.f;
        if (eff > best_eff * 1.02f) { best_eff = eff; best_nc = nc; }
    }
    q.nc = best_nc;
    q.cw = (st + q.nc - 1) / q.nc;
    int G = 32 / q.cw; if (G > ngr) G = ngr; if (G < 1) G = 1;
    int wc_cap = kWarps;
    for (;;) {
        const int slots = (ngr + G - 1) / G;                 // row-warps that have work
        int WR = 1; while (WR < slots && WR < kWarps) WR <<= 1;
        int WC = kWarps / WR;
        while (WC > 1 && (WC > q.nc || WC > wc_cap || WC * q.cw > kMaxColsT)) WC >>= 1;
        q.G = G; q.WR = WR; q.WC = WC;
        q.RT = WR * G * kA;
        q.rows = q.RT + q.MB - 1;
        q.colsT = WC * q.cw;
        q.pitch = q.colsT;
        if (G > 1)
            for (int p = q.colsT; p < q.colsT + 16; ++p) if (pitch_ok(p, G, q.cw)) { q.pitch = p; break; }
        const int xs = q.rows * q.pitch, gs = q.MB * q.colsT, tot = q.npass * q.WC * q.RT;
        if (2 * xs + 2 * gs + tot <= kSmemDoubles || (G == 1 && wc_cap == 1)) {
            q.xs_off[0] = 0; q.xs_off[1] = xs;
            q.gs_off[0] = 2 * xs; q.gs_off[1] = 2 * xs + gs;
            q.tot_off = 2 * xs + 2 * gs;
            break;
        }
        if (G > 1) --G; else wc_cap >>= 1;
    }
    q.nrt = (q.nW + q.RT - 1) / q.RT;
    q.nccs = (q.nc + q.WC - 1) / q.WC;
}

// A x MB outer-product walk: 35 X loads + 21 template loads feed 315 FMAs (MB = 21).
template <int MB>
__device__ __forceinline__ void rows_fma(const double* __restrict__ xs, int pitch,
                                         const double* __restrict__ gs, int gp, double (&acc)[kA]) {
    double g[MB];
#pragma unroll
    for (int m = 0; m < MB; ++m) { g[m] = *gs; gs += gp; }
#pragma unroll
    for (int gam = 0; gam < kA + MB - 1; ++gam) {
        const double x = *xs;
        xs += pitch;
#pragma unroll
        for (int al = 0; al < kA; ++al) {
            const int m = gam - al;
            if (m >= 0 && m < MB) acc[al] = fma(g[m], x, acc[al]);
        }
    }
}

}  // namespace

namespace {

template <bool UNIFORM>
__global__ void __launch_bounds__(kThreads, 2) k_chi2_rows(TileArgs a) {
    extern __shared__ double smem[];
    __shared__ Geom s_q;
    __shared__ Cand s_best[kWarps];
    __shared__ double s_tmpl[kTmplSmem];

    const int jd = blockIdx.x, pl = blockIdx.y;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const DurEntry e = a.durtab[(long long)pl * a.n_dur + jd];
    Partial* out = a.partial + (long long)pl * a.n_dur + jd;
    if (e.skip) {
        if (tid == 0) { out->valid = 0; out->dchi2 = 0.0; out->depth = 0.0; out->start = 0; }
        return;
    }
    if (tid == 0) make_geom(s_q, a.n, e.D, e.stride, a.n_tmpl, UNIFORM);
    const bool tmpl_in_smem = a.n_tmpl <= kTmplSmem;
    if (tmpl_in_smem) for (int k = tid; k < a.n_tmpl; k += kThreads) s_tmpl[k] = a.tmpl[k];
    const double* __restrict__ tm = tmpl_in_smem ? s_tmpl : a.tmpl;
    __syncthreads();
    const Geom& q = s_q;
    // fields used inside loops are copied to registers (shared memory would be re-read after
    // every barrier); the rest is read from s_q once per stage
    const int D = q.D, st = q.st, g_pitch = q.pitch, g_colsT = q.colsT, g_rows = q.rows,
              g_MB = q.MB, g_cw = q.cw, g_WC = q.WC, g_nc = q.nc;
    const double g_tscale = q.tscale;
    const double* __restrict__ x1 = a.x1 + (long long)pl * a.pitch;
    const double* __restrict__ x0 = a.x0 + (long long)pl * a.pitch;
    const double* __restrict__ s1 = a.s1 + (long long)pl * a.spitch;
    const double* __restrict__ s0 = a.s0 + (long long)pl * a.spitch;
    const long long lim = (long long)a.n + D;          // x entries >= lim are never needed
    const double G_u = a.w_uniform * e.gg2, sw_u = (double)D * a.w_uniform;

    // loader role: thread -> (row offset, staged column)
    const int ld_rpp = kThreads / q.colsT;             // rows copied per sweep
    const int ld_r0 = tid / q.colsT, ld_col = tid - ld_r0 * q.colsT;
    const int ld_wc = ld_col / q.cw, ld_c = ld_col - ld_wc * q.cw;
    const bool ld_on = ld_r0 < ld_rpp;
    const int ld_iters = ld_on ? (g_rows - ld_r0 + ld_rpp - 1) / ld_rpp : 0;   // rows this thread copies
    // compute role: warp -> (wr, wc), lane -> (g, c)
    const int wr = warp / q.WC, wc = warp - wr * q.WC;
    const int lg = lane / q.cw, lc = lane - lg * q.cw;
    const bool cmp_on = warp < q.WR * q.WC && lane < q.G * q.cw;
    const int grp = wr * q.G + lg;                      // window group inside the row tile

    auto issue_stage = [&](int rt, int pass, int ccs, int mb, int buf) {
        double* XS = smem + q.xs_off[buf];
        double* GS = smem + q.gs_off[buf];
        const double* __restrict__ src = (UNIFORM || pass == 0) ? x1 : x0;
        const long long row0 = (long long)rt * q.RT + (long long)mb * g_MB;
        if (ld_on) {
            const int cc = ccs * g_WC + ld_wc;
            const int i = cc * g_cw + ld_c;
            const bool colv = cc < g_nc && i < st;
            const long long ee = (row0 + ld_r0) * st + i;
            const long long estep = (long long)ld_rpp * st;
            const double* sp = src + ee;
            unsigned dst = (unsigned)__cvta_generic_to_shared(XS + ld_r0 * g_pitch + ld_col);
            const unsigned dstep = (unsigned)(ld_rpp * g_pitch * 8);
            // rows of this thread's column that lie inside the curve come first, then zero fill
            int nvalid = 0;
            if (colv && ee < lim) {
                const long long nv = (lim - ee + estep - 1) / estep;
                nvalid = nv > ld_iters ? ld_iters : (int)nv;
            }
            int k = 0;
            for (; k < nvalid; ++k) { cp_async8(dst, sp, true); sp += estep; dst += dstep; }
            for (; k < ld_iters; ++k) { cp_async8(dst, src, false); dst += dstep; }
            // template values of the same column, rows m = ld_r0, ld_r0 + ld_rpp, ...
            double* gd = GS + ld_r0 * g_colsT + ld_col;
            const int gstep = ld_rpp * g_colsT;
            long long j = (long long)(mb * g_MB + ld_r0) * st + i;
            for (int m = ld_r0; m < g_MB; m += ld_rpp) {
                double gv = 0.0;
                if (colv && j < D) {
                    const double u = ((double)(int)j + 0.5) * g_tscale;
                    int kk = (int)u;                       // u >= 0: truncation == floor
                    kk = kk > a.n_tmpl - 2 ? a.n_tmpl - 2 : kk;
                    const double fr = u - (double)kk;
                    const double t0 = tm[kk];
                    gv = t0 + fr * (tm[kk + 1] - t0);
                    if (!UNIFORM && pass == 1) gv *= gv;
                }
                *gd = gv;
                gd += gstep; j += estep;
            }
        }
        cp_async_commit();
    };

    Cand best; best.has = 0; best.d = 0.0; best.s = 0; best.depth = 0.0;
    double acc[kA];
    const int stages_per_pass = q.nccs * q.nmb;
    const int stages_per_rt = q.npass * stages_per_pass;
    const int S = q.nrt * stages_per_rt;
    // stage counters (rt, pass, ccs, mb) of the stage being computed / being issued
    int c_rt = 0, c_pass = 0, c_ccs = 0, c_mb = 0;
    int n_rt = 0, n_pass = 0, n_ccs = 0, n_mb = 0;
    auto advance = [&](int& rt, int& pass, int& ccs, int& mb) {
        if (++mb == q.nmb) { mb = 0; if (++ccs == q.nccs) { ccs = 0; if (++pass == q.npass) { pass = 0; ++rt; } } }
    };
    issue_stage(0, 0, 0, 0, 0);
    advance(n_rt, n_pass, n_ccs, n_mb);

    for (int s = 0; s < S; ++s) {
        const int buf = s & 1;
        // stage s has landed for every thread; everyone is also done reading the other buffer
        cp_async_wait<0>();
        __syncthreads();
        if (s + 1 < S) {      // staging of stage s+1 overlaps the FMAs of stage s (no barrier between)
            issue_stage(n_rt, n_pass, n_ccs, n_mb, buf ^ 1);
            advance(n_rt, n_pass, n_ccs, n_mb);
        }
        if (c_ccs == 0 && c_mb == 0) {
#pragma unroll
            for (int al = 0; al < kA; ++al) acc[al] = 0.0;
        }
        if (cmp_on) {
            const double* xs = smem + q.xs_off[buf] + (grp * kA) * g_pitch + wc * g_cw + lc;
            const double* gs = smem + q.gs_off[buf] + wc * g_cw + lc;
            if (g_MB == 21) rows_fma<21>(xs, g_pitch, gs, g_colsT, acc);
            else if (g_MB == 14) rows_fma<14>(xs, g_pitch, gs, g_colsT, acc);
            else rows_fma<7>(xs, g_pitch, gs, g_colsT, acc);
        }
        const bool end_pass = (c_ccs == q.nccs - 1) && (c_mb == q.nmb - 1);
        if (end_pass) {
            // segmented reduction over the cw lanes of each window group
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) {
#pragma unroll
                for (int al = 0; al < kA; ++al) {
                    const double v = __shfl_down_sync(0xffffffffu, acc[al], off);
                    if (lc + off < g_cw) acc[al] += v;
                }
            }
            if (cmp_on && lc == 0) {
                double* tot = smem + q.tot_off + (c_pass * q.WC + wc) * q.RT + grp * kA;
#pragma unroll
                for (int al = 0; al < kA; ++al) tot[al] = acc[al];
            }
            if (c_pass == q.npass - 1) {          // row tile complete: a5 + a8 per window
                __syncthreads();
                const double* tot = smem + q.tot_off;
                for (int w = tid; w < q.RT; w += kThreads) {
                    const int k = c_rt * q.RT + w;
                    if (k >= q.nW) continue;
                    double C = 0.0, Gs = 0.0;
                    for (int c2 = 0; c2 < q.WC; ++c2) {
                        C += tot[c2 * q.RT + w];
                        if (!UNIFORM) Gs += tot[(q.WC + c2) * q.RT + w];
                    }
                    const int sidx = k * st;
                    const double swr = s1[sidx + D] - s1[sidx];
                    const double sw = UNIFORM ? sw_u : s0[sidx + D] - s0[sidx];
                    const double rbar = __ddiv_rn(swr, sw);
                    const double depth = __ddiv_rn(fmax(rbar, 0.0), e.gbar);
                    const double Gv = UNIFORM ? G_u : Gs;
                    const double d = -2.0 * depth * C + (depth * depth) * Gv;
                    cand_offer(best, d, sidx, depth);
                }
            }
        }
        advance(c_rt, c_pass, c_ccs, c_mb);      // the barrier at the top of the next stage orders buffer reuse
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
        for (int k = 1; k < kWarps; ++k)
            if (s_best[k].has) cand_offer(best, s_best[k].d, s_best[k].s, s_best[k].depth);
        out->valid = best.has; out->dchi2 = best.d; out->depth = best.depth; out->start = best.s;
    }
}

}  // namespace

void launch_chi2_rows(const TileArgs& a, cudaStream_t st) {
    const dim3 grid(a.n_dur, a.tile);
    const size_t sm = (size_t)kSmemDoubles * sizeof(double);
    static bool set = false;
    if (!set) {
        cudaFuncSetAttribute(k_chi2_rows<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
        cudaFuncSetAttribute(k_chi2_rows<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
        set = true;
    }
    if (a.uniform) k_chi2_rows<true><<<grid, kThreads, sm, st>>>(a);
    else k_chi2_rows<false><<<grid, kThreads, sm, st>>>(a);
}

}  // namespace gtls
