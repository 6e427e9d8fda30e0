// Steps a1-a4 fused, fast path: fold (Eq. 10) -> stable phase sort (ties by
// original index) -> gather + wrap pad (Fig. 3) -> prefix sums (Eq. 14)
// with two HBM passes over 8-byte keys instead of the ten of the LSD radix path (fold_sort.cu +
// scan.cu, kept as the fallback):
//
//   k_bucket_count    fold every point; one histogram of the top KBITS bits of floor(phase * 2^32) per CTA
//                     (2048 points), written out as 16-bit counts -- no global atomics
//   k_bucket_scan     per period: for every bucket the running sum of the CTAs' counts (where a CTA's keys
//                     start inside the bucket) and the bucket starts; a bucket larger than kBucketCap
//                     (clustered phases) puts the period on the tile's fallback list, which the LSD path
//                     processes instead
//   k_bucket_scatter  fold again (t is L2 resident, the division is cheaper than 16 B of HBM) and write
//                     (key32 << 32 | index) to bucket start + CTA offset + rank inside the CTA's share
//                     (shared-memory atomics only; the CTA's keys are staged in bucket order in shared
//                     memory and written by consecutive threads; any order inside the bucket)
//   k_bucket_sort     one WARP per (period, 8 consecutive buckets of ~260 keys) with warp-private shared memory
//                     and no CTA barrier: counting sort on the next 8 key bits, an exact rank inside every run
//                     of equal 8-bit codes by (key32, fp64 phase, index), then the permutation and the gathered
//                     x1 = w r (x0 = w, x2 = w r^2) go out coalesced.  Units are independent, so periods with
//                     clustered phases (long runs) are balanced over the GPU by the CTA scheduler.
//   k_bucket_prefix   one CTA per period: S1 (S0, S2) over the n sorted entries and on over the wrap padding
//                     (Fig. 3: the first D_m sorted entries again), coalesced, fixed addition tree.
//
// The order inside a bucket before the local sort is irrelevant because the local sort orders by the
// full (phase, index) key, so the permutation is identical to a stable sort by fp64 phase
// (bit-exact against the oracle) and the prefix sums are deterministic (fixed addition tree).
#include "gtls_internal.cuh"

namespace gtls {

namespace {

constexpr int kCountThreads = 256;
constexpr int kCountItems = 8;                       // points per thread in count / scatter
constexpr int kCtaKeys = kCountThreads * kCountItems;   // 2048 points per CTA (a 16-bit count holds it)
constexpr int kFinWarps = 4;                         // periods per CTA of the finish kernel
constexpr int kFinSlots = kBucketCap / 32;           // keys per lane and bucket (12)
constexpr int kUnitsPerWarp = 8;                     // consecutive buckets of a period a warp sorts (<= 31)
constexpr int kPrefThreads = 256, kPrefItems = 8;    // prefix-sum kernel: 2048 entries per chunk
#ifndef GTLS_SUB_BITS
#define GTLS_SUB_BITS 8
#endif
constexpr int kSubBits = GTLS_SUB_BITS;
constexpr int kSub = 1 << kSubBits;                  // sub-buckets of the warp's counting sort
static_assert(kSub % 128 == 0, "sort: whole uint4 groups of counts per lane");
static_assert(kBucketCap % 32 == 0 && kCtaKeys < 65536, "bucket slots / 16-bit counts");
static_assert(kMaxBuckets % kCountThreads == 0, "scatter: whole buckets per thread in the scan");

// (A reciprocal-multiply quotient with two residual corrections and an exact-residual check that proves it equal
//  to the IEEE quotient was measured in place of the division: the folds got slower, DESIGN.md section 10 item 4.)
__device__ __forceinline__ u32 key32_of(double t, double period) {
    return phase_key32(fold_phase(t, period));
}

__global__ void __launch_bounds__(kCountThreads) k_bucket_count(BucketArgs b) {
    __shared__ u32 h[kMaxBuckets];
    const int pl = blockIdx.y;
    for (int k = threadIdx.x; k < b.nbk; k += kCountThreads) h[k] = 0;
    __syncthreads();
    const double period = b.periods[b.p0 + pl];
    const int base = blockIdx.x * kCtaKeys + threadIdx.x;
    double tv[kCountItems];
#pragma unroll
    for (int e = 0; e < kCountItems; ++e) tv[e] = base + e * kCountThreads < b.n ? b.t[base + e * kCountThreads] : 0.0;
#pragma unroll
    for (int e = 0; e < kCountItems; ++e) {
        const u32 key = key32_of(tv[e], period);
        if (base + e * kCountThreads < b.n) atomicAdd(&h[(u32)((u64)key >> b.shift)], 1u);
    }
    __syncthreads();
    unsigned short* hist = b.hist + ((long long)pl * b.ncta + blockIdx.x) * b.nbk;
    for (int k = threadIdx.x; k < b.nbk; k += kCountThreads) hist[k] = (unsigned short)h[k];
}

// one CTA per period: where every CTA's keys start inside every bucket, the bucket starts, the overflow flag
__global__ void __launch_bounds__(256) k_bucket_scan(BucketArgs b) {
    __shared__ u32 tot[kMaxBuckets];
    __shared__ u32 s_big[8];
    const int pl = blockIdx.x, tid = threadIdx.x, lane = tid & 31;
    const unsigned short* hist = b.hist + (long long)pl * b.ncta * b.nbk;
    u32* rel = b.rel + (long long)pl * b.ncta * b.nbk;
    u32 big = 0;
    for (int k = tid; k < b.nbk; k += 256) {
        u32 run = 0;
        for (int c = 0; c < b.ncta; ++c) {
            const u32 h = hist[(long long)c * b.nbk + k];
            rel[(long long)c * b.nbk + k] = run;
            run += h;
        }
        tot[k] = run;
        big = max(big, run);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) big = max(big, __shfl_xor_sync(0xffffffffu, big, o));
    if (lane == 0) s_big[tid >> 5] = big;
    __syncthreads();
    if (tid >= 32) return;
    u32* start = b.start + (long long)pl * (b.nbk + 1);
    u32 carry = 0;
    for (int k0 = 0; k0 < b.nbk; k0 += 32) {
        const int k = k0 + lane;
        const u32 c = k < b.nbk ? tot[k] : 0;
        u32 x = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const u32 y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
        if (k < b.nbk) start[k] = carry + x - c;
        carry += __shfl_sync(0xffffffffu, x, 31);
    }
    if (lane == 0) {
        start[b.nbk] = carry;
        big = 0;
        for (int k = 0; k < 8; ++k) big = max(big, s_big[k]);
        const int over = big > (u32)kBucketCap ? 1 : 0;
        b.fb_flag[pl] = over;
        if (over) b.fb_list[atomicAdd(b.fb_count, 1)] = pl;
    }
}

// The CTA's 2048 keys are put in bucket order in shared memory first (their rank inside the CTA's share of a
// bucket comes from the histogram atomics), then written out by consecutive threads: a warp's 32 stores fall
// into four or five runs of consecutive addresses instead of 32 buckets (the kernel is bound by L2 write
// transactions otherwise).
__global__ void __launch_bounds__(kCountThreads) k_bucket_scatter(BucketArgs b) {
    extern __shared__ __align__(16) unsigned char scat_smem[];
    u64* const stage = reinterpret_cast<u64*>(scat_smem);                 // [kCtaKeys]
    u32* const cnt = reinterpret_cast<u32*>(stage + kCtaKeys);            // [nbk] keys of this CTA per bucket, then the bucket's first staged position
    u32* const basepos = cnt + b.nbk;                                     // [nbk] bucket start + where this CTA's keys start inside the bucket
    __shared__ u32 s_wsum[kCountThreads / 32];
    const int pl = blockIdx.y;
    if (b.fb_flag[pl]) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    {
        const u32* start = b.start + (long long)pl * (b.nbk + 1);
        const u32* rel = b.rel + ((long long)pl * b.ncta + blockIdx.x) * b.nbk;
        for (int k = tid; k < b.nbk; k += kCountThreads) { cnt[k] = 0; basepos[k] = start[k] + rel[k]; }
    }
    __syncthreads();
    const double period = b.periods[b.p0 + pl];
    const int base = blockIdx.x * kCtaKeys + tid;
    // all loads, then all folds, then the ranks (the atomics would otherwise keep the items in line)
    double tv[kCountItems];
#pragma unroll
    for (int e = 0; e < kCountItems; ++e) tv[e] = base + e * kCountThreads < b.n ? b.t[base + e * kCountThreads] : 0.0;
    u32 key[kCountItems], rank[kCountItems];
#pragma unroll
    for (int e = 0; e < kCountItems; ++e) key[e] = key32_of(tv[e], period);
#pragma unroll
    for (int e = 0; e < kCountItems; ++e)
        rank[e] = base + e * kCountThreads < b.n ? atomicAdd(&cnt[(u32)((u64)key[e] >> b.shift)], 1u) : 0u;
    __syncthreads();
    // exclusive scan of the counts (kMaxBuckets / kCountThreads consecutive buckets per thread)
    {
        constexpr int PER = kMaxBuckets / kCountThreads;
        u32 c[PER], sum = 0;
#pragma unroll
        for (int k = 0; k < PER; ++k) { c[k] = tid * PER + k < b.nbk ? cnt[tid * PER + k] : 0u; sum += c[k]; }
        u32 x = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const u32 y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
        if (lane == 31) s_wsum[warp] = x;
        __syncthreads();
        u32 wb = 0;
#pragma unroll
        for (int k = 0; k < kCountThreads / 32; ++k) wb += k < warp ? s_wsum[k] : 0u;
        u32 run = wb + x - sum;
#pragma unroll
        for (int k = 0; k < PER; ++k) { if (tid * PER + k < b.nbk) cnt[tid * PER + k] = run; run += c[k]; }
    }
    __syncthreads();
#pragma unroll
    for (int e = 0; e < kCountItems; ++e)
        if (base + e * kCountThreads < b.n)
            stage[cnt[(u32)((u64)key[e] >> b.shift)] + rank[e]] = ((u64)key[e] << 32) | (u64)(u32)(base + e * kCountThreads);
    __syncthreads();
    const int total = min(kCtaKeys, b.n - (int)blockIdx.x * kCtaKeys);
    u64* dst = b.keys + (long long)pl * b.n;
#pragma unroll
    for (int e = 0; e < kCountItems; ++e) {
        const int i = e * kCountThreads + tid;
        if (i < total) {
            const u64 k = stage[i];
            const u32 bk = (u32)((k >> 32) >> b.shift);
            dst[basepos[bk] + ((u32)i - cnt[bk])] = k;
        }
    }
}

// strict total order (key32, fp64 phase, index) == (fp64 phase, index)
__device__ __forceinline__ bool key_less(const u64 a, const u64 b, const double* __restrict__ t,
                                         const double period) {
    const u32 ka = (u32)(a >> 32), kb = (u32)(b >> 32);
    if (ka != kb) return ka < kb;
    const double pa = fold_phase(t[(u32)a], period), pb = fold_phase(t[(u32)b], period);
    if (pa != pb) return pa < pb;
    return (u32)a < (u32)b;
}

// warp-private scratch of the sort kernel
struct FinWarp {
    u64 B[kBucketCap];          // keys in sub-bucket order; afterwards the doubles of the gather / scan
    u32 A[kBucketCap];          // point indices in sorted order
    u32 H[kSub + 8];            // counts -> starts -> (after the scatter) ends of the sub-buckets
};

// rare: two keys of a run share their 32-bit key, the fp64 phases decide (kept out of line)
__device__ __noinline__ int rank_by_phase(const u64* B, int rs, int re, int i, const double* __restrict__ t, double period) {
    const u64 k = B[i];
    int r = rs;
    for (int j = rs; j < re; ++j) r += (j != i && key_less(B[j], k, t, period)) ? 1 : 0;
    return r;
}

// One WARP per (period, bucket) unit, kUnitsPerWarp consecutive buckets of a period per warp: warp-private shared
// memory, no CTA barrier, and the units are independent (the prefix sums are a kernel of their own), so the
// hardware balances periods with clustered phases (long runs of equal 8-bit codes) over the whole GPU.
template <bool HAS0, bool HAS2, bool SORT_ONLY>
__global__ void __launch_bounds__(kFinWarps * 32, 7) k_bucket_sort(BucketArgs b) {
    __shared__ __align__(16) FinWarp sm_all[kFinWarps];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int gpp = (b.nbk + kUnitsPerWarp - 1) / kUnitsPerWarp;            // bucket groups per period
    const long long g = (long long)blockIdx.x * kFinWarps + warp;
    if (g >= (long long)b.tile * gpp) return;
    const int pl = (int)(g / gpp), bk0 = (int)(g % gpp) * kUnitsPerWarp;
    if (b.fb_flag[pl]) return;
    FinWarp& sm = sm_all[warp];
    const double period = b.periods[b.p0 + pl];
    const u32* start = b.start + (long long)pl * (b.nbk + 1);
    const u64* keys = b.keys + (long long)pl * b.n;
    const int subshift = b.shift - kSubBits;                   // sub-bucket = next kSubBits key bits
    u32* perm = b.perm + (long long)pl * b.n;
    double* x1 = b.x1 + (long long)pl * b.pitch;
    double* x0 = HAS0 ? b.x0 + (long long)pl * b.pitch : nullptr;
    double* x2 = HAS2 ? b.x2 + (long long)pl * b.pitch : nullptr;
#pragma unroll
    for (int k = 0; k < kSub / 32; ++k) sm.H[k * 32 + lane] = 0;
    __syncwarp();
    const u32 bounds = start[min(bk0 + lane, b.nbk)];          // starts of the group's buckets (and the end of the last)
    const int nb = min(kUnitsPerWarp, b.nbk - bk0);
    for (int u = 0; u < nb; ++u) {
        const int bs = (int)__shfl_sync(0xffffffffu, bounds, u), be = (int)__shfl_sync(0xffffffffu, bounds, u + 1);
        const int M = be - bs;
        if (M == 0) continue;
        // 1. + 2. keys (entry j * 32 + lane), histogram of the next 8 key bits (H is all zero here)
        u64 kc[kFinSlots];
        {
            const u64* const kp = keys + bs + lane;
#pragma unroll
            for (int j = 0; j < kFinSlots; ++j) kc[j] = j * 32 + lane < M ? kp[j * 32] : 0ull;
#pragma unroll
            for (int j = 0; j < kFinSlots; ++j)
                if (j * 32 + lane < M) atomicAdd(&sm.H[((u32)(kc[j] >> 32) >> subshift) & (kSub - 1)], 1u);
        }
        __syncwarp();
        // 3. exclusive scan of the kSub counts (kSub / 32 consecutive counts per lane)
        {
            constexpr int PB = kSub / 32;
            u32 c[PB], sum = 0;
#pragma unroll
            for (int q = 0; q < PB / 4; ++q) {
                const uint4 v = *reinterpret_cast<const uint4*>(&sm.H[lane * PB + 4 * q]);
                c[4 * q] = v.x; c[4 * q + 1] = v.y; c[4 * q + 2] = v.z; c[4 * q + 3] = v.w;
                sum += v.x + v.y + v.z + v.w;
            }
            u32 x = sum;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const u32 y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
            u32 base = x - sum;
#pragma unroll
            for (int q = 0; q < PB / 4; ++q) {
                uint4 v;
                v.x = base; base += c[4 * q]; v.y = base; base += c[4 * q + 1];
                v.z = base; base += c[4 * q + 2]; v.w = base; base += c[4 * q + 3];
                *reinterpret_cast<uint4*>(&sm.H[lane * PB + 4 * q]) = v;
            }
        }
        __syncwarp();
        // 4. counting-sort scatter (order inside a sub-bucket is arbitrary)
#pragma unroll
        for (int j = 0; j < kFinSlots; ++j)
            if (j * 32 + lane < M) sm.B[atomicAdd(&sm.H[((u32)(kc[j] >> 32) >> subshift) & (kSub - 1)], 1u)] = kc[j];
        __syncwarp();
        // 5. exact rank inside every run of equal 8-bit codes (a run of one ranks itself): (key32, index) orders
        //    the run unless two of its 32-bit keys are equal
#pragma unroll 1
        for (int i = lane; i < M; i += 32) {
            const u64 k = sm.B[i];
            const u32 sb = ((u32)(k >> 32) >> subshift) & (kSub - 1);
            const int rs = sb ? (int)sm.H[sb - 1] : 0, re = (int)sm.H[sb];     // H[sb] is now the end of sub-bucket sb
            int r = rs, same = 0;
#pragma unroll 1
            for (int j = rs; j < re; ++j) {
                const u64 o = sm.B[j];
                r += o < k ? 1 : 0;
                same += (u32)(o >> 32) == (u32)(k >> 32) ? 1 : 0;
            }
            if (same > 1) r = rank_by_phase(sm.B, rs, re, i, b.t, period);
            sm.A[r] = (u32)k;
        }
        __syncwarp();
#pragma unroll
        for (int k = 0; k < kSub / 32; ++k) sm.H[k * 32 + lane] = 0;   // for the next bucket (ordered by the barrier below)
        // 6. the bucket is sorted: permutation and the gathered arrays, coalesced
#pragma unroll
        for (int j = 0; j < kFinSlots; ++j) {
            const int i = j * 32 + lane;
            if (i < M) {
                const u32 idx = sm.A[i];
                perm[bs + i] = idx;
                if (!SORT_ONLY) {
                    x1[bs + i] = b.wr[idx];
                    if (HAS0) x0[bs + i] = b.w[idx];
                    if (HAS2) x2[bs + i] = b.wr2[idx];
                }
            }
        }
        __syncwarp();                                                  // A, B, H are reused by the next bucket
    }
}

// a4 (Eq. 14): S[i + 1] = x[0] + .. + x[i] for the n sorted entries of every period; one CTA per period walks
// the period in chunks of 2048 entries.  A warp owns 256 consecutive entries of the chunk: it loads and stores
// them lane-strided (coalesced; the next chunk's loads are issued before the current chunk is scanned) and
// turns them through a padded warp-private tile of shared memory so that a lane scans 8 consecutive entries;
// the warps' totals meet in shared memory, a running carry links the chunks.  Fixed addition tree.
template <int NARR>
__global__ void __launch_bounds__(kPrefThreads) k_bucket_prefix(BucketArgs b) {
    constexpr int NW = kPrefThreads / 32, WE = 32 * kPrefItems, CH = kPrefThreads * kPrefItems;
    __shared__ double s_t[NW][WE + WE / 8];
    __shared__ double s_w[2][NARR][NW];
    const int pl = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (b.fb_flag[pl]) return;
    double* xs[3] = {b.x1 + (long long)pl * b.pitch, NARR > 1 ? b.x0 + (long long)pl * b.pitch : nullptr,
                     NARR > 2 ? b.x2 + (long long)pl * b.pitch : nullptr};
    // wrap padding (Fig. 3): entries n .. n + pad - 1 repeat entries 0 .. pad - 1 and the sums run on
    int pad = b.pad_override;
    if (pad < 0) {
        pad = 0;
        for (int jd = 0; jd < b.n_dur; ++jd) pad = max(pad, b.durtab[(long long)pl * b.n_dur + jd].D);
    }
    const int nt = b.n + pad;
    double* ss[3] = {b.s1 + (long long)pl * b.spitch, NARR > 1 ? b.s0 + (long long)pl * b.spitch : nullptr,
                     NARR > 2 ? b.s2 + (long long)pl * b.spitch : nullptr};
    double carry[NARR];
#pragma unroll
    for (int a = 0; a < NARR; ++a) { carry[a] = 0.0; if (tid == 0) ss[a][0] = 0.0; }
    double nx[NARR][kPrefItems];
    double* const T = s_t[warp];
    auto load = [&](int c0) {
        const int g = c0 + warp * WE + lane;
#pragma unroll
        for (int a = 0; a < NARR; ++a)
#pragma unroll
            for (int e = 0; e < kPrefItems; ++e) {
                const int i = g + e * 32;
                if (c0 + CH <= b.n) {                                    // (CTA uniform) loads only: all in flight at once
                    nx[a][e] = __ldg(xs[a] + i);
                } else {
                    nx[a][e] = i < nt ? xs[a][i < b.n ? i : i - b.n] : 0.0;
                    if (i >= b.n && i < nt) xs[a][i] = nx[a][e];
                }
            }
    };
    load(0);
    int par = 0;
    for (int c0 = 0; c0 < nt; c0 += CH, par ^= 1) {
        double v[NARR][kPrefItems], tot[NARR], incl[NARR];
#pragma unroll
        for (int a = 0; a < NARR; ++a) {
            // lane-strided -> 8 consecutive entries per lane (tile index j + j / 8: conflict-free both ways)
#pragma unroll
            for (int e = 0; e < kPrefItems; ++e) { const int j = e * 32 + lane; T[j + (j >> 3)] = nx[a][e]; }
            __syncwarp();
#pragma unroll
            for (int e = 0; e < kPrefItems; ++e) v[a][e] = T[lane * (kPrefItems + 1) + e];
            __syncwarp();
        }
        if (c0 + CH < nt) load(c0 + CH);
#pragma unroll
        for (int a = 0; a < NARR; ++a) {
#pragma unroll
            for (int e = 1; e < kPrefItems; ++e) v[a][e] += v[a][e - 1];
            tot[a] = v[a][kPrefItems - 1];
            incl[a] = tot[a];
        }
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
#pragma unroll
            for (int a = 0; a < NARR; ++a) {
                const double u = __shfl_up_sync(0xffffffffu, incl[a], o);
                if (lane >= o) incl[a] += u;
            }
        }
        if (lane == 31) {
#pragma unroll
            for (int a = 0; a < NARR; ++a) s_w[par][a][warp] = incl[a];
        }
        __syncthreads();                                               // (s_w is double buffered: one barrier per chunk)
        const int g = c0 + warp * WE + lane;
#pragma unroll
        for (int a = 0; a < NARR; ++a) {
            double w = carry[a], all = carry[a];
#pragma unroll
            for (int k = 0; k < NW; ++k) { const double x = s_w[par][a][k]; if (k < warp) w += x; all += x; }
            const double off = w + (incl[a] - tot[a]);
#pragma unroll
            for (int e = 0; e < kPrefItems; ++e) T[lane * (kPrefItems + 1) + e] = off + v[a][e];
            __syncwarp();
            double* dst = ss[a] + g + 1;
#pragma unroll
            for (int e = 0; e < kPrefItems; ++e) {
                const int j = e * 32 + lane;
                if (g + e * 32 < nt) dst[e * 32] = T[j + (j >> 3)];
            }
            __syncwarp();
            carry[a] = all;
        }
    }
}

}  // namespace

int bucket_count_for(int n) {
    int nbk = 1;
    while (nbk < kMaxBuckets && (n + nbk - 1) / nbk > kBucketTarget) nbk <<= 1;
    return nbk;
}

static dim3 count_grid(const BucketArgs& b) { return dim3(b.ncta, b.tile); }
static size_t scatter_smem(const BucketArgs& b) { return kCtaKeys * sizeof(u64) + 2 * (size_t)b.nbk * sizeof(u32); }

int bucket_cta_count(int n) { return (n + kCtaKeys - 1) / kCtaKeys; }

void launch_bucket_sort_head(const BucketArgs& b, cudaStream_t st) {
    cudaMemsetAsync(b.fb_count, 0, sizeof(int), st);
    k_bucket_count<<<count_grid(b), kCountThreads, 0, st>>>(b);
    k_bucket_scan<<<b.tile, 256, 0, st>>>(b);
}

void launch_bucket_sort_tail(const BucketArgs& b, bool has0, bool has2, bool sort_only, cudaStream_t st) {
    // (per device and cheap: set on every call)
    cudaFuncSetAttribute(k_bucket_scatter, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)scatter_smem(b));
    k_bucket_scatter<<<count_grid(b), kCountThreads, scatter_smem(b), st>>>(b);
    const long long groups = (long long)b.tile * ((b.nbk + kUnitsPerWarp - 1) / kUnitsPerWarp);
    const dim3 fgrid((unsigned)((groups + kFinWarps - 1) / kFinWarps));
    constexpr int kFinThreads = kFinWarps * 32;
    if (sort_only) { k_bucket_sort<false, false, true><<<fgrid, kFinThreads, 0, st>>>(b); return; }
    if (has2) {
        k_bucket_sort<true, true, false><<<fgrid, kFinThreads, 0, st>>>(b);
        k_bucket_prefix<3><<<b.tile, kPrefThreads, 0, st>>>(b);
    } else if (has0) {
        k_bucket_sort<true, false, false><<<fgrid, kFinThreads, 0, st>>>(b);
        k_bucket_prefix<2><<<b.tile, kPrefThreads, 0, st>>>(b);
    } else {
        k_bucket_sort<false, false, false><<<fgrid, kFinThreads, 0, st>>>(b);
        k_bucket_prefix<1><<<b.tile, kPrefThreads, 0, st>>>(b);
    }
}

}  // namespace gtls
