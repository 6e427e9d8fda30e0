// Steps a1-a4 fused, fast path: fold (Eq. 10) -> stable phase sort (ties by
// original index) -> gather + wrap pad (Fig. 3) -> prefix sums (Eq. 14)
// with two HBM passes over 8-byte keys instead of the ten of the LSD radix path (fold_sort.cu +
// scan.cu, kept as the fallback):
//
//   k_bucket_count    fold every point; one histogram of the top KBITS bits of floor(phase * 2^32) per CTA
//                     (4096 points), written out as 16-bit counts -- no global atomics
//   k_bucket_scan     per period: for every bucket the running sum of the CTAs' counts (where a CTA's keys
//                     start inside the bucket) and the bucket starts; a bucket larger than kBucketCap
//                     (clustered phases) puts the period on the tile's fallback list, which the LSD path
//                     processes instead
//   k_bucket_scatter  fold again (t is L2 resident, the division is cheaper than 16 B of HBM) and write
//                     (key32 << 32 | index) to bucket start + CTA offset + rank inside the CTA's share
//                     (shared-memory atomics only; any order inside the bucket)
//   k_bucket_finish   one WARP per period walks through the period's buckets (~260 keys each) in order,
//                     with warp-private shared memory and no CTA barrier: counting sort on the next 8 key
//                     bits, an exact rank inside every run of equal 8-bit codes by (key32, fp64 phase,
//                     index), then gather and scan with the running sums carried from bucket to bucket:
//                     permutation, x1 = w r (x0 = w) and the final S1 (S0) in one pass, every global
//                     access coalesced.
//   k_pad_scan        wrap padding (Fig. 3): the first D_m sorted entries again, the sums run on.
//
// The order inside a bucket before the local sort is irrelevant because the local sort orders by the
// full (phase, index) key, so the permutation is identical to a stable sort by fp64 phase
// (bit-exact against the oracle) and the prefix sums are deterministic (fixed addition tree).
#include "gtls_internal.cuh"

namespace gtls {

namespace {

constexpr int kCountThreads = 512;
constexpr int kCountItems = 8;                       // points per thread in count / scatter
constexpr int kCtaKeys = kCountThreads * kCountItems;   // 4096 points per CTA (a 16-bit count holds it)
constexpr int kFinWarps = 4;                         // periods per CTA of the finish kernel
constexpr int kFinSlots = kBucketCap / 32;           // keys per lane and bucket (12)
constexpr int kUnitsPerWarp = 8;                     // consecutive buckets of a period a warp sorts (<= 31)
constexpr int kPrefThreads = 512, kPrefItems = 8;    // prefix-sum kernel: 4096 entries per chunk
constexpr int kPadThreads = 512;
constexpr int kSubBits = 8;
constexpr int kSub = 1 << kSubBits;                  // sub-buckets of the warp's counting sort
constexpr int kScanItems = 4;                        // pad scan: entries per thread and round
static_assert(kBucketCap % 32 == 0 && kCtaKeys < 65536, "bucket slots / 16-bit counts");
static_assert(kMaxBuckets % kCountThreads == 0, "scatter: whole buckets per thread in the scan");

__device__ __forceinline__ u32 key32_of(const double* __restrict__ t, int i, double period) {
    return phase_key32(fold_phase(t[i], period));
}

__global__ void __launch_bounds__(kCountThreads) k_bucket_count(BucketArgs b) {
    __shared__ u32 h[kMaxBuckets];
    const int pl = blockIdx.y;
    for (int k = threadIdx.x; k < b.nbk; k += kCountThreads) h[k] = 0;
    __syncthreads();
    const double period = b.periods[b.p0 + pl];
    const int base = blockIdx.x * kCtaKeys;
#pragma unroll
    for (int e = 0; e < kCountItems; ++e) {
        const int i = base + e * kCountThreads + threadIdx.x;
        if (i < b.n) atomicAdd(&h[(u32)((u64)key32_of(b.t, i, period) >> b.shift)], 1u);
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

// The CTA's 4096 keys are put in bucket order in shared memory first (their rank inside the CTA's share of a
// bucket comes from the histogram atomics), then written out by consecutive threads: a warp's 32 stores fall
// into four or five runs of consecutive addresses instead of 32 buckets (the kernel is bound by L2 write
// transactions otherwise).
__global__ void __launch_bounds__(kCountThreads) k_bucket_scatter(BucketArgs b) {
    extern __shared__ __align__(16) unsigned char scat_smem[];
    u64* const stage = reinterpret_cast<u64*>(scat_smem);                 // [kCtaKeys]
    __shared__ u32 cnt[kMaxBuckets];           // keys of this CTA per bucket, then the bucket's first staged position
    __shared__ u32 basepos[kMaxBuckets];       // bucket start + where this CTA's keys start inside the bucket
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
    for (int e = 0; e < kCountItems; ++e) key[e] = phase_key32(fold_phase(tv[e], period));
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
        // 3. exclusive scan of the kSub counts (8 per lane)
        {
            uint4 c0 = *reinterpret_cast<const uint4*>(&sm.H[lane * 8]);
            uint4 c1 = *reinterpret_cast<const uint4*>(&sm.H[lane * 8 + 4]);
            const u32 sum = c0.x + c0.y + c0.z + c0.w + c1.x + c1.y + c1.z + c1.w;
            u32 x = sum;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const u32 y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
            u32 base = x - sum;
            uint4 e0, e1;
            e0.x = base; base += c0.x; e0.y = base; base += c0.y; e0.z = base; base += c0.z; e0.w = base; base += c0.w;
            e1.x = base; base += c1.x; e1.y = base; base += c1.y; e1.z = base; base += c1.z; e1.w = base;
            *reinterpret_cast<uint4*>(&sm.H[lane * 8]) = e0;
            *reinterpret_cast<uint4*>(&sm.H[lane * 8 + 4]) = e1;
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
// the period in chunks of 4096 entries.  A warp owns 256 consecutive entries of the chunk: it loads and stores
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
    const double* xs[3] = {b.x1 + (long long)pl * b.pitch, NARR > 1 ? b.x0 + (long long)pl * b.pitch : nullptr,
                           NARR > 2 ? b.x2 + (long long)pl * b.pitch : nullptr};
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
            for (int e = 0; e < kPrefItems; ++e) nx[a][e] = g + e * 32 < b.n ? xs[a][g + e * 32] : 0.0;
    };
    load(0);
    int par = 0;
    for (int c0 = 0; c0 < b.n; c0 += CH, par ^= 1) {
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
        if (c0 + CH < b.n) load(c0 + CH);
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
                if (g + e * 32 < b.n) dst[e * 32] = T[j + (j >> 3)];
            }
            __syncwarp();
            carry[a] = all;
        }
    }
}

// Wrap padding (Fig. 3): entries n .. n+pad-1 repeat entries 0 .. pad-1, the prefix sums run on.
template <bool HAS0, bool HAS2>
__global__ void __launch_bounds__(kPadThreads) k_pad_scan(BucketArgs b) {
    __shared__ double s_w[3][32];
    const int pl = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (b.fb_flag[pl]) return;
    constexpr int NW = kPadThreads / 32;
    int pad = b.pad_override;
    if (pad < 0) {
        pad = 0;
        for (int jd = 0; jd < b.n_dur; ++jd) pad = max(pad, b.durtab[(long long)pl * b.n_dur + jd].D);
    }
    double* x1 = b.x1 + (long long)pl * b.pitch;
    double* s1 = b.s1 + (long long)pl * b.spitch;
    double* x0 = HAS0 ? b.x0 + (long long)pl * b.pitch : nullptr;
    double* s0 = HAS0 ? b.s0 + (long long)pl * b.spitch : nullptr;
    double* x2 = HAS2 ? b.x2 + (long long)pl * b.pitch : nullptr;
    double* s2 = HAS2 ? b.s2 + (long long)pl * b.spitch : nullptr;
    double c1 = s1[b.n], c0 = HAS0 ? s0[b.n] : 0.0, c2 = HAS2 ? s2[b.n] : 0.0;
    for (int r0 = 0; r0 < pad; r0 += kPadThreads * kScanItems) {
        const int cnt = min(kPadThreads * kScanItems, pad - r0);
        double v1[kScanItems], v0[kScanItems], v2[kScanItems];
        const int first = threadIdx.x * kScanItems;
#pragma unroll
        for (int e = 0; e < kScanItems; ++e) {
            v1[e] = 0.0; v0[e] = 0.0; v2[e] = 0.0;
            if (first + e < cnt) {
                v1[e] = x1[r0 + first + e];
                x1[b.n + r0 + first + e] = v1[e];
                if (HAS0) { v0[e] = x0[r0 + first + e]; x0[b.n + r0 + first + e] = v0[e]; }
                if (HAS2) { v2[e] = x2[r0 + first + e]; x2[b.n + r0 + first + e] = v2[e]; }
            }
        }
#pragma unroll
        for (int e = 1; e < kScanItems; ++e) { v1[e] += v1[e - 1]; v0[e] += v0[e - 1]; v2[e] += v2[e - 1]; }
        double t1 = v1[kScanItems - 1], t0 = v0[kScanItems - 1], t2 = v2[kScanItems - 1];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const double u1 = __shfl_up_sync(0xffffffffu, t1, o);
            const double u0 = __shfl_up_sync(0xffffffffu, t0, o);
            const double u2 = __shfl_up_sync(0xffffffffu, t2, o);
            if (lane >= o) { t1 += u1; t0 += u0; t2 += u2; }
        }
        if (lane == 31) { s_w[0][warp] = t1; s_w[1][warp] = t0; s_w[2][warp] = t2; }
        __syncthreads();
        double w1 = c1, w0 = c0, w2 = c2, a1 = c1, a0 = c0, a2 = c2;
#pragma unroll
        for (int k = 0; k < NW; ++k) {
            if (k < warp) { w1 += s_w[0][k]; w0 += s_w[1][k]; w2 += s_w[2][k]; }
            a1 += s_w[0][k]; a0 += s_w[1][k]; a2 += s_w[2][k];
        }
        const double o1 = w1 + (t1 - v1[kScanItems - 1]), o0 = w0 + (t0 - v0[kScanItems - 1]),
                     o2 = w2 + (t2 - v2[kScanItems - 1]);
#pragma unroll
        for (int e = 0; e < kScanItems; ++e) {
            if (first + e < cnt) {
                s1[b.n + r0 + first + e + 1] = o1 + v1[e];
                if (HAS0) s0[b.n + r0 + first + e + 1] = o0 + v0[e];
                if (HAS2) s2[b.n + r0 + first + e + 1] = o2 + v2[e];
            }
        }
        c1 = a1; c0 = a0; c2 = a2;
        __syncthreads();
    }
}

}  // namespace

int bucket_count_for(int n) {
    int nbk = 1;
    while (nbk < kMaxBuckets && (n + nbk - 1) / nbk > kBucketTarget) nbk <<= 1;
    return nbk;
}

static dim3 count_grid(const BucketArgs& b) { return dim3(b.ncta, b.tile); }

int bucket_cta_count(int n) { return (n + kCtaKeys - 1) / kCtaKeys; }

void launch_bucket_sort_head(const BucketArgs& b, cudaStream_t st) {
    cudaMemsetAsync(b.fb_count, 0, sizeof(int), st);
    k_bucket_count<<<count_grid(b), kCountThreads, 0, st>>>(b);
    k_bucket_scan<<<b.tile, 256, 0, st>>>(b);
}

void launch_bucket_sort_tail(const BucketArgs& b, bool has0, bool has2, bool sort_only, cudaStream_t st) {
    // (per device and cheap: set on every call)
    cudaFuncSetAttribute(k_bucket_scatter, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kCtaKeys * sizeof(u64)));
    k_bucket_scatter<<<count_grid(b), kCountThreads, kCtaKeys * sizeof(u64), st>>>(b);
    const long long groups = (long long)b.tile * ((b.nbk + kUnitsPerWarp - 1) / kUnitsPerWarp);
    const dim3 fgrid((unsigned)((groups + kFinWarps - 1) / kFinWarps));
    constexpr int kFinThreads = kFinWarps * 32;
    if (sort_only) { k_bucket_sort<false, false, true><<<fgrid, kFinThreads, 0, st>>>(b); return; }
    if (has2) {
        k_bucket_sort<true, true, false><<<fgrid, kFinThreads, 0, st>>>(b);
        k_bucket_prefix<3><<<b.tile, kPrefThreads, 0, st>>>(b);
        k_pad_scan<true, true><<<b.tile, kPadThreads, 0, st>>>(b);
    } else if (has0) {
        k_bucket_sort<true, false, false><<<fgrid, kFinThreads, 0, st>>>(b);
        k_bucket_prefix<2><<<b.tile, kPrefThreads, 0, st>>>(b);
        k_pad_scan<true, false><<<b.tile, kPadThreads, 0, st>>>(b);
    } else {
        k_bucket_sort<false, false, false><<<fgrid, kFinThreads, 0, st>>>(b);
        k_bucket_prefix<1><<<b.tile, kPrefThreads, 0, st>>>(b);
        k_pad_scan<false, false><<<b.tile, kPadThreads, 0, st>>>(b);
    }
}

}  // namespace gtls
