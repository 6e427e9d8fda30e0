// Steps a1-a4 fused, fast path: fold (Eq. 10) -> stable phase sort (ties by
// original index) -> gather + wrap pad (Fig. 3) -> prefix sums (Eq. 14)
// with two HBM passes over 8-byte keys instead of the ten of the LSD radix path (fold_sort.cu +
// scan.cu, kept as the fallback):
//
//   k_bucket_count    fold every point, histogram of the top KBITS bits of floor(phase * 2^32)
//   k_bucket_scan     per period: bucket starts; a bucket larger than kBucketCap (clustered phases) puts
//                     the period on the tile's fallback list, which the LSD path processes instead
//   k_bucket_scatter  fold again (t is L2 resident, the division is cheaper than 16 B of HBM) and
//                     write (key32 << 32 | index) into its bucket, any order inside the bucket
//   k_bucket_finish   one CTA per period walks through its buckets in order: a bucket (~1000 keys) is
//                     sorted entirely in shared memory -- counting sort on the next 10 key bits, then an
//                     exact rank inside every run of equal 10-bit codes by (key32, fp64 phase, index) --
//                     gathered and scanned with the running sums carried from bucket to bucket:
//                     permutation, x1 = w r (x0 = w) and the final S1 (S0) in one pass.
//   k_pad_scan        wrap padding (Fig. 3): the first D_m sorted entries again, the sums run on.
//
// The order inside a bucket before the local sort is irrelevant because the local sort orders by the
// full (phase, index) key, so the permutation is identical to a stable sort by fp64 phase
// (bit-exact against the oracle) and the prefix sums are deterministic (fixed addition tree).
#include "gtls_internal.cuh"

namespace gtls {

namespace {

constexpr int kCountThreads = 256;
constexpr int kCountItems = 8;                       // points per thread in count / scatter
#ifndef GTLS_FIN_CTAS
#define GTLS_FIN_CTAS 4
#endif
constexpr int kFinCtas = GTLS_FIN_CTAS;              // resident CTAs per SM the finish kernel is compiled for
#ifndef GTLS_FIN_THREADS
#define GTLS_FIN_THREADS 256
#endif
constexpr int kFinThreads = GTLS_FIN_THREADS;                     // one CTA per period
constexpr int kFinItems = kBucketCap / kFinThreads;  // sorted entries per thread (6)
constexpr int kPadThreads = 512;
#ifndef GTLS_SUB_BITS
#define GTLS_SUB_BITS 10
#endif
constexpr int kSubBits = GTLS_SUB_BITS;
constexpr int kSub = 1 << kSubBits;                  // sub-buckets of the local counting sort
constexpr int kScanItems = 4;                        // pad scan: entries per thread and round

__device__ __forceinline__ u32 key32_of(const double* __restrict__ t, int i, double period) {
    return phase_key32(fold_phase(t[i], period));
}

__global__ void __launch_bounds__(kCountThreads) k_bucket_count(BucketArgs b) {
    __shared__ u32 h[kMaxBuckets];
    const int pl = blockIdx.y;
    for (int k = threadIdx.x; k < b.nbk; k += kCountThreads) h[k] = 0;
    __syncthreads();
    const double period = b.periods[b.p0 + pl];
    const int base = blockIdx.x * (kCountThreads * kCountItems);
#pragma unroll
    for (int e = 0; e < kCountItems; ++e) {
        const int i = base + e * kCountThreads + threadIdx.x;
        if (i < b.n) atomicAdd(&h[(u32)((u64)key32_of(b.t, i, period) >> b.shift)], 1u);
    }
    __syncthreads();
    u32* hist = b.hist + (long long)pl * b.nbk;
    for (int k = threadIdx.x; k < b.nbk; k += kCountThreads)
        if (h[k]) atomicAdd(&hist[k], h[k]);
}

// one warp per period: exclusive scan of the bucket histogram, cursors, overflow flag
__global__ void __launch_bounds__(256) k_bucket_scan(BucketArgs b) {
    const int pl = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (pl >= b.tile) return;
    const u32* hist = b.hist + (long long)pl * b.nbk;
    u32* start = b.start + (long long)pl * (b.nbk + 1);
    u32* cursor = b.cursor + (long long)pl * b.nbk;
    u32 carry = 0, big = 0;
    for (int k0 = 0; k0 < b.nbk; k0 += 32) {
        const int k = k0 + lane;
        const u32 c = k < b.nbk ? hist[k] : 0;
        big = max(big, c);
        u32 x = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const u32 y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
        if (k < b.nbk) { start[k] = carry + x - c; cursor[k] = carry + x - c; }
        carry += __shfl_sync(0xffffffffu, x, 31);
    }
    if (lane == 0) start[b.nbk] = carry;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) big = max(big, __shfl_xor_sync(0xffffffffu, big, o));
    if (lane == 0) {
        const int over = big > (u32)kBucketCap ? 1 : 0;
        b.fb_flag[pl] = over;
        if (over) b.fb_list[atomicAdd(b.fb_count, 1)] = pl;
    }
}

__global__ void __launch_bounds__(kCountThreads) k_bucket_scatter(BucketArgs b) {
    __shared__ u32 cnt[kMaxBuckets];
    __shared__ u32 basepos[kMaxBuckets];
    const int pl = blockIdx.y;
    if (b.fb_flag[pl]) return;
    for (int k = threadIdx.x; k < b.nbk; k += kCountThreads) cnt[k] = 0;
    __syncthreads();
    const double period = b.periods[b.p0 + pl];
    const int base = blockIdx.x * (kCountThreads * kCountItems);
    u32 key[kCountItems], rank[kCountItems];
#pragma unroll
    for (int e = 0; e < kCountItems; ++e) {
        const int i = base + e * kCountThreads + threadIdx.x;
        key[e] = 0; rank[e] = 0;
        if (i < b.n) {
            key[e] = key32_of(b.t, i, period);
            rank[e] = atomicAdd(&cnt[(u32)((u64)key[e] >> b.shift)], 1u);
        }
    }
    __syncthreads();
    u32* cursor = b.cursor + (long long)pl * b.nbk;
    for (int k = threadIdx.x; k < b.nbk; k += kCountThreads)
        basepos[k] = cnt[k] ? atomicAdd(&cursor[k], cnt[k]) : 0u;
    __syncthreads();
    u64* dst = b.keys + (long long)pl * b.n;
#pragma unroll
    for (int e = 0; e < kCountItems; ++e) {
        const int i = base + e * kCountThreads + threadIdx.x;
        if (i < b.n) dst[basepos[(u32)((u64)key[e] >> b.shift)] + rank[e]] = ((u64)key[e] << 32) | (u64)(u32)i;
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

// One CTA per PERIOD walks through the period's buckets in order, so the running prefix sums are carried
// in registers from bucket to bucket (no look-back between CTAs, no second pass over S1), the next
// bucket's keys are already on their way while the current bucket is sorted, and the per-CTA set-up is
// paid once per period.
template <bool HAS0, bool HAS2, bool SORT_ONLY>
__global__ void __launch_bounds__(kFinThreads, kFinCtas) k_bucket_finish(BucketArgs b) {
    extern __shared__ __align__(16) unsigned char fin_smem[];
    u64* const A = reinterpret_cast<u64*>(fin_smem);           // [kBucketCap]
    u64* const B = A + kBucketCap;                             // [kBucketCap]
    u32* const H = reinterpret_cast<u32*>(B + kBucketCap);     // [kSub + 1] counts -> starts -> (after the scatter) ends
    __shared__ double s_w[3][kFinThreads / 32];
    __shared__ u32 s_wsum[kFinThreads / 32];
    const int pl = blockIdx.x;
    if (b.fb_flag[pl]) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = kFinThreads / 32;
    const double period = b.periods[b.p0 + pl];
    const u32* start = b.start + (long long)pl * (b.nbk + 1);
    const u64* keys = b.keys + (long long)pl * b.n;
    const int subshift = b.shift - kSubBits;                   // sub-bucket = next kSubBits key bits
    u32* perm = b.perm + (long long)pl * b.n;
    double* x1 = b.x1 + (long long)pl * b.pitch;
    double* x0 = HAS0 ? b.x0 + (long long)pl * b.pitch : nullptr;
    double* x2 = HAS2 ? b.x2 + (long long)pl * b.pitch : nullptr;
    double* s1 = b.s1 + (long long)pl * b.spitch;
    double* s0 = HAS0 ? b.s0 + (long long)pl * b.spitch : nullptr;
    double* s2 = HAS2 ? b.s2 + (long long)pl * b.spitch : nullptr;
    if (!SORT_ONLY && tid == 0) { s1[0] = 0.0; if (HAS0) s0[0] = 0.0; if (HAS2) s2[0] = 0.0; }
    double carry1 = 0.0, carry0 = 0.0, carry2 = 0.0;           // sums of the buckets before the current one

    // keys of the first bucket
    u64 nk[kFinItems];
    int bs = (int)start[0], be = (int)start[1];
#pragma unroll
    for (int e = 0; e < kFinItems; ++e) {
        const int i = e * kFinThreads + tid;
        nk[e] = bs + i < be ? keys[bs + i] : 0ull;
    }
    for (int bk = 0; bk < b.nbk; ++bk) {
        const int m = be - bs;
        // 1. the prefetched keys stay in registers (thread owns entries e*kFinThreads + tid); the next
        //    bucket's keys are requested
        u64 kc[kFinItems];
#pragma unroll
        for (int e = 0; e < kFinItems; ++e) kc[e] = nk[e];
        for (int k = tid; k < kSub; k += kFinThreads) H[k] = 0;
        const int nbs = be, nbe = bk + 1 < b.nbk ? (int)start[bk + 2] : be;
#pragma unroll
        for (int e = 0; e < kFinItems; ++e) {
            const int i = e * kFinThreads + tid;
            nk[e] = nbs + i < nbe ? keys[nbs + i] : 0ull;
        }
        __syncthreads();
        // 2. histogram of the next 10 key bits
#pragma unroll
        for (int e = 0; e < kFinItems; ++e)
            if (e * kFinThreads + tid < m) atomicAdd(&H[((u32)(kc[e] >> 32) >> subshift) & (kSub - 1)], 1u);
        __syncthreads();
        // 3. exclusive scan of the kSub counts (4 per thread)
        {
            constexpr int PER = kSub / kFinThreads;
            u32 c[PER], sum = 0;
#pragma unroll
            for (int e = 0; e < PER; ++e) { c[e] = H[tid * PER + e]; sum += c[e]; }
            u32 x = sum;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const u32 y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
            if (lane == 31) s_wsum[warp] = x;
            __syncthreads();
            u32 wbase = 0;
#pragma unroll
            for (int k = 0; k < NW; ++k) wbase += k < warp ? s_wsum[k] : 0u;
            u32 base = wbase + x - sum;
#pragma unroll
            for (int e = 0; e < PER; ++e) { H[tid * PER + e] = base; base += c[e]; }
        }
        __syncthreads();
        // 4. counting-sort scatter (order inside a sub-bucket is arbitrary)
        {
            u32 pos[kFinItems];
#pragma unroll
            for (int e = 0; e < kFinItems; ++e)
                pos[e] = e * kFinThreads + tid < m
                             ? atomicAdd(&H[((u32)(kc[e] >> 32) >> subshift) & (kSub - 1)], 1u) : 0u;
#pragma unroll
            for (int e = 0; e < kFinItems; ++e)
                if (e * kFinThreads + tid < m) B[pos[e]] = kc[e];
        }
        __syncthreads();
        // 5. exact rank inside every run of equal 10-bit codes
        for (int i = tid; i < m; i += kFinThreads) {
            const u64 k = B[i];
            const u32 sb = ((u32)(k >> 32) >> subshift) & (kSub - 1);
            const int rs = sb ? (int)H[sb - 1] : 0, re = (int)H[sb];     // H[sb] is now the end of sub-bucket sb
            int r = i;
            if (re - rs > 1) {
                // (key32, index) orders the run unless two of its 32-bit keys are equal: then (rare) the
                // fp64 phases decide
                r = rs;
                bool tie = false;
                for (int j = rs; j < re; ++j) {
                    const u64 o = B[j];
                    r += o < k ? 1 : 0;
                    tie |= j != i && (u32)(o >> 32) == (u32)(k >> 32);
                }
                if (tie) {
                    r = rs;
                    for (int j = rs; j < re; ++j) r += (j != i && key_less(B[j], k, b.t, period)) ? 1 : 0;
                }
            }
            A[r] = k;
        }
        __syncthreads();
        // 6. the bucket is sorted: permutation
        for (int i = tid; i < m; i += kFinThreads) perm[bs + i] = (u32)A[i];
        if (!SORT_ONLY) {
            // 7. gather + inclusive scan: thread owns kFinItems consecutive sorted entries
            double v1[kFinItems], v0[kFinItems], v2[kFinItems];
            const int first = tid * kFinItems;
#pragma unroll
            for (int e = 0; e < kFinItems; ++e) {
                v1[e] = 0.0; v0[e] = 0.0; v2[e] = 0.0;
                if (first + e < m) {
                    const u32 idx = (u32)A[first + e];
                    v1[e] = b.wr[idx];
                    if (HAS0) v0[e] = b.w[idx];
                    if (HAS2) v2[e] = b.wr2[idx];
                }
            }
#pragma unroll
            for (int e = 0; e < kFinItems; ++e) {
                if (first + e < m) {
                    x1[bs + first + e] = v1[e];
                    if (HAS0) x0[bs + first + e] = v0[e];
                    if (HAS2) x2[bs + first + e] = v2[e];
                }
            }
#pragma unroll
            for (int e = 1; e < kFinItems; ++e) {
                v1[e] += v1[e - 1];
                if (HAS0) v0[e] += v0[e - 1];
                if (HAS2) v2[e] += v2[e - 1];
            }
            double t1 = v1[kFinItems - 1], t0 = v0[kFinItems - 1], t2 = v2[kFinItems - 1];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const double u1 = __shfl_up_sync(0xffffffffu, t1, o);
                const double u0 = HAS0 ? __shfl_up_sync(0xffffffffu, t0, o) : 0.0;
                const double u2 = HAS2 ? __shfl_up_sync(0xffffffffu, t2, o) : 0.0;
                if (lane >= o) { t1 += u1; t0 += u0; t2 += u2; }
            }
            if (lane == 31) { s_w[0][warp] = t1; s_w[1][warp] = t0; s_w[2][warp] = t2; }
            __syncthreads();
            // carry + totals of the warps before mine (every thread adds in the same fixed order)
            double w1 = carry1, w0 = carry0, w2 = carry2, a1 = carry1, a0 = carry0, a2 = carry2;
#pragma unroll
            for (int k = 0; k < NW; ++k) {
                if (k < warp) { w1 += s_w[0][k]; w0 += s_w[1][k]; w2 += s_w[2][k]; }
                a1 += s_w[0][k]; a0 += s_w[1][k]; a2 += s_w[2][k];
            }
            const double o1 = w1 + (t1 - v1[kFinItems - 1]);
            const double o0 = w0 + (t0 - v0[kFinItems - 1]);
            const double o2 = w2 + (t2 - v2[kFinItems - 1]);
#pragma unroll
            for (int e = 0; e < kFinItems; ++e) {
                if (first + e < m) {
                    s1[bs + first + e + 1] = o1 + v1[e];
                    if (HAS0) s0[bs + first + e + 1] = o0 + v0[e];
                    if (HAS2) s2[bs + first + e + 1] = o2 + v2[e];
                }
            }
            carry1 = a1; carry0 = a0; carry2 = a2;
        }
        bs = nbs; be = nbe;
        __syncthreads();                                           // A, H, s_w are reused by the next bucket
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

constexpr size_t kFinSmem = 2 * (size_t)kBucketCap * sizeof(u64) + (kSub + 1) * sizeof(u32);

static dim3 count_grid(const BucketArgs& b) {
    return dim3((b.n + kCountThreads * kCountItems - 1) / (kCountThreads * kCountItems), b.tile);
}

void launch_bucket_sort_head(const BucketArgs& b, cudaStream_t st) {
    cudaMemsetAsync(b.hist, 0, (size_t)b.tile * b.nbk * sizeof(u32), st);
    cudaMemsetAsync(b.fb_count, 0, sizeof(int), st);
    k_bucket_count<<<count_grid(b), kCountThreads, 0, st>>>(b);
    k_bucket_scan<<<(b.tile * 32 + 255) / 256, 256, 0, st>>>(b);
}

void launch_bucket_sort_tail(const BucketArgs& b, bool has0, bool has2, bool sort_only, cudaStream_t st) {
    {   // per device and cheap: set on every call (a process-wide flag would miss a second device)
        cudaFuncSetAttribute(k_bucket_finish<false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFinSmem);
        cudaFuncSetAttribute(k_bucket_finish<true, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFinSmem);
        cudaFuncSetAttribute(k_bucket_finish<true, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFinSmem);
        cudaFuncSetAttribute(k_bucket_finish<false, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFinSmem);
    }
    k_bucket_scatter<<<count_grid(b), kCountThreads, 0, st>>>(b);
    const dim3 fgrid(b.tile);
    if (sort_only) { k_bucket_finish<false, false, true><<<fgrid, kFinThreads, kFinSmem, st>>>(b); return; }
    if (has2) {
        k_bucket_finish<true, true, false><<<fgrid, kFinThreads, kFinSmem, st>>>(b);
        k_pad_scan<true, true><<<b.tile, kPadThreads, 0, st>>>(b);
    } else if (has0) {
        k_bucket_finish<true, false, false><<<fgrid, kFinThreads, kFinSmem, st>>>(b);
        k_pad_scan<true, false><<<b.tile, kPadThreads, 0, st>>>(b);
    } else {
        k_bucket_finish<false, false, false><<<fgrid, kFinThreads, kFinSmem, st>>>(b);
        k_pad_scan<false, false><<<b.tile, kPadThreads, 0, st>>>(b);
    }
}

}  // namespace gtls
