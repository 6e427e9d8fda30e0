// Steps a1-a4 fused, fast path: fold (Eq. 10) -> stable phase sort (ties by
// original index) -> gather + wrap pad (Fig. 3) -> prefix sums (Eq. 14)
// with two HBM passes over 8-byte keys instead of the ten of the LSD radix path (fold_sort.cu +
// scan.cu, kept as the fallback):
//
//   k_bucket_count    fold every point, histogram of the top KBITS bits of floor(phase * 2^32)
//   k_bucket_scan     per period: bucket starts; a bucket larger than kBucketCap raises the tile's
//                     fallback flag (clustered phases), and the LSD path redoes the whole tile
//   k_bucket_scatter  fold again (t is L2 resident, the division is cheaper than 16 B of HBM) and
//                     write (key32 << 32 | index) into its bucket, any order inside the bucket
//   k_bucket_finish   one CTA per period walks its buckets in phase order; each bucket (~2000 keys)
//                     is sorted entirely in shared memory -- counting sort on the next 12 key bits,
//                     then an exact rank inside every run of equal 12-bit codes by
//                     (key32, fp64 phase, index) -- and is gathered, scanned and written straight
//                     from shared memory: permutation, x1 = w r (x0 = w), S1 (S0).
//
// The order inside a bucket before the local sort is irrelevant because the local sort orders by the
// full (phase, index) key, so the permutation is identical to a stable sort by fp64 phase
// (bit-exact against the oracle) and the prefix sums are deterministic (fixed addition tree).
#include "gtls_internal.cuh"

namespace gtls {

namespace {

constexpr int kCountThreads = 256;
constexpr int kCountItems = 8;                       // points per thread in count / scatter
constexpr int kFinThreads = 512;
constexpr int kSubBits = 12;
constexpr int kSub = 1 << kSubBits;                  // sub-buckets of the local counting sort
constexpr int kScanItems = 4;                        // entries per thread and scan round

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
    if (lane == 0 && (big > (u32)kBucketCap || b.force_fallback)) atomicExch(b.fallback, 1);
}

__global__ void __launch_bounds__(kCountThreads) k_bucket_scatter(BucketArgs b) {
    __shared__ u32 cnt[kMaxBuckets];
    __shared__ u32 basepos[kMaxBuckets];
    if (*b.fallback) return;
    const int pl = blockIdx.y;
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

struct ScanState {                 // running carries of the (up to three) prefix sums of one period
    double c1, c0, c2;
};

// One scan round over `cnt` (<= kFinThreads * kScanItems) consecutive entries starting at padded
// position pos0: thread-local scan of 4 entries, warp shuffles, warp totals through shared memory.
template <bool HAS0, bool HAS2, typename Fetch>
__device__ __forceinline__ void scan_round(const int cnt, const long long pos0, Fetch fetch,
                                           double* __restrict__ x1, double* __restrict__ s1,
                                           double* __restrict__ x0, double* __restrict__ s0,
                                           double* __restrict__ x2, double* __restrict__ s2,
                                           double (*s_w)[32], ScanState& st) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    constexpr int NW = kFinThreads / 32;
    double v1[kScanItems], v0[kScanItems], v2[kScanItems];
    const int first = threadIdx.x * kScanItems;
#pragma unroll
    for (int e = 0; e < kScanItems; ++e) {
        v1[e] = 0.0; v0[e] = 0.0; v2[e] = 0.0;
        if (first + e < cnt) {
            fetch(first + e, v1[e], v0[e], v2[e]);
            x1[pos0 + first + e] = v1[e];
            if (HAS0) x0[pos0 + first + e] = v0[e];
            if (HAS2) x2[pos0 + first + e] = v2[e];
        }
    }
#pragma unroll
    for (int e = 1; e < kScanItems; ++e) {
        v1[e] += v1[e - 1];
        if (HAS0) v0[e] += v0[e - 1];
        if (HAS2) v2[e] += v2[e - 1];
    }
    double t1 = v1[kScanItems - 1], t0 = v0[kScanItems - 1], t2 = v2[kScanItems - 1];
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const double u1 = __shfl_up_sync(0xffffffffu, t1, o);
        const double u0 = HAS0 ? __shfl_up_sync(0xffffffffu, t0, o) : 0.0;
        const double u2 = HAS2 ? __shfl_up_sync(0xffffffffu, t2, o) : 0.0;
        if (lane >= o) { t1 += u1; t0 += u0; t2 += u2; }
    }
    if (lane == 31) { s_w[0][warp] = t1; s_w[1][warp] = t0; s_w[2][warp] = t2; }
    __syncthreads();
    if (warp == 0) {
        double w1 = lane < NW ? s_w[0][lane] : 0.0, w0 = lane < NW ? s_w[1][lane] : 0.0,
               w2 = lane < NW ? s_w[2][lane] : 0.0;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const double u1 = __shfl_up_sync(0xffffffffu, w1, o);
            const double u0 = __shfl_up_sync(0xffffffffu, w0, o);
            const double u2 = __shfl_up_sync(0xffffffffu, w2, o);
            if (lane >= o) { w1 += u1; w0 += u0; w2 += u2; }
        }
        s_w[0][lane] = w1; s_w[1][lane] = w0; s_w[2][lane] = w2;
    }
    __syncthreads();
    const double b1 = st.c1 + (warp ? s_w[0][warp - 1] : 0.0) + (t1 - v1[kScanItems - 1]);
    const double b0 = HAS0 ? st.c0 + (warp ? s_w[1][warp - 1] : 0.0) + (t0 - v0[kScanItems - 1]) : 0.0;
    const double b2 = HAS2 ? st.c2 + (warp ? s_w[2][warp - 1] : 0.0) + (t2 - v2[kScanItems - 1]) : 0.0;
#pragma unroll
    for (int e = 0; e < kScanItems; ++e) {
        if (first + e < cnt) {
            s1[pos0 + first + e + 1] = b1 + v1[e];
            if (HAS0) s0[pos0 + first + e + 1] = b0 + v0[e];
            if (HAS2) s2[pos0 + first + e + 1] = b2 + v2[e];
        }
    }
    st.c1 += s_w[0][31];
    if (HAS0) st.c0 += s_w[1][31];
    if (HAS2) st.c2 += s_w[2][31];
    __syncthreads();
}

template <bool HAS0, bool HAS2, bool SORT_ONLY>
__global__ void __launch_bounds__(kFinThreads) k_bucket_finish(BucketArgs b) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    u64* A = reinterpret_cast<u64*>(smem_raw);                 // [kBucketCap]
    u64* B = A + kBucketCap;                                   // [kBucketCap]
    u32* H = reinterpret_cast<u32*>(B + kBucketCap);           // [kSub + 1] counts -> starts
    u32* cur = H + kSub + 1;                                   // [kSub]
    __shared__ double s_w[3][32];
    __shared__ u32 s_wsum[kFinThreads / 32];
    if (*b.fallback) return;
    const int pl = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const double period = b.periods[b.p0 + pl];
    const u64* keys = b.keys + (long long)pl * b.n;
    const u32* start = b.start + (long long)pl * (b.nbk + 1);
    u32* perm = b.perm + (long long)pl * b.n;
    double* x1 = SORT_ONLY ? nullptr : b.x1 + (long long)pl * b.pitch;
    double* s1 = SORT_ONLY ? nullptr : b.s1 + (long long)pl * b.spitch;
    double* x0 = HAS0 ? b.x0 + (long long)pl * b.pitch : nullptr;
    double* s0 = HAS0 ? b.s0 + (long long)pl * b.spitch : nullptr;
    double* x2 = HAS2 ? b.x2 + (long long)pl * b.pitch : nullptr;
    double* s2 = HAS2 ? b.s2 + (long long)pl * b.spitch : nullptr;
    ScanState st; st.c1 = st.c0 = st.c2 = 0.0;
    if (!SORT_ONLY && tid == 0) { s1[0] = 0.0; if (HAS0) s0[0] = 0.0; if (HAS2) s2[0] = 0.0; }
    const int subshift = b.shift - kSubBits;                   // sub-bucket = next kSubBits key bits

    for (int bk = 0; bk < b.nbk; ++bk) {
        const int bs = (int)start[bk], m = (int)start[bk + 1] - bs;
        if (m == 0) continue;
        // 1. load the bucket, clear the sub-bucket histogram
        for (int i = tid; i < m; i += kFinThreads) A[i] = keys[bs + i];
        for (int k = tid; k <= kSub; k += kFinThreads) H[k] = 0;
        __syncthreads();
        // 2. histogram of the next 12 key bits
        for (int i = tid; i < m; i += kFinThreads)
            atomicAdd(&H[((u32)(A[i] >> 32) >> subshift) & (kSub - 1)], 1u);
        __syncthreads();
        // 3. exclusive scan of the kSub counts (8 per thread)
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
            if (warp == 0) {
                u32 w = lane < kFinThreads / 32 ? s_wsum[lane] : 0, y0 = w;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) { const u32 y = __shfl_up_sync(0xffffffffu, y0, o); if (lane >= o) y0 += y; }
                if (lane < kFinThreads / 32) s_wsum[lane] = y0 - w;
            }
            __syncthreads();
            u32 base = s_wsum[warp] + x - sum;
#pragma unroll
            for (int e = 0; e < PER; ++e) { H[tid * PER + e] = base; cur[tid * PER + e] = base; base += c[e]; }
            if (tid == kFinThreads - 1) H[kSub] = base;
        }
        __syncthreads();
        // 4. counting-sort scatter (order inside a sub-bucket is arbitrary)
        for (int i = tid; i < m; i += kFinThreads) {
            const u64 k = A[i];
            B[atomicAdd(&cur[((u32)(k >> 32) >> subshift) & (kSub - 1)], 1u)] = k;
        }
        __syncthreads();
        // 5. exact rank inside every run of equal 12-bit codes
        for (int i = tid; i < m; i += kFinThreads) {
            const u64 k = B[i];
            const u32 sb = ((u32)(k >> 32) >> subshift) & (kSub - 1);
            const int rs = (int)H[sb], re = (int)H[sb + 1];
            int r = i;
            if (re - rs > 1) {
                r = rs;
                for (int j = rs; j < re; ++j) r += (j != i && key_less(B[j], k, b.t, period)) ? 1 : 0;
            }
            A[r] = k;
        }
        __syncthreads();
        // 6. the bucket is sorted: permutation, gather, scan
        for (int i = tid; i < m; i += kFinThreads) perm[bs + i] = (u32)A[i];
        if (!SORT_ONLY) {
            for (int r0 = 0; r0 < m; r0 += kFinThreads * kScanItems) {
                auto fetch = [&](int e, double& v1, double& v0, double& v2) {
                    const u32 idx = (u32)A[r0 + e];
                    v1 = b.wr[idx];
                    if (HAS0) v0 = b.w[idx];
                    if (HAS2) v2 = b.wr2[idx];
                };
                scan_round<HAS0, HAS2>(min(kFinThreads * kScanItems, m - r0), (long long)bs + r0, fetch,
                                       x1, s1, x0, s0, x2, s2, s_w, st);
            }
        }
        __syncthreads();
    }
    if (SORT_ONLY) return;
    // wrap padding (Fig. 3): the first `pad` sorted entries again, the sums run on
    int pad = b.pad_override;
    if (pad < 0) {
        pad = 0;
        for (int jd = 0; jd < b.n_dur; ++jd) pad = max(pad, b.durtab[(long long)pl * b.n_dur + jd].D);
    }
    for (int r0 = 0; r0 < pad; r0 += kFinThreads * kScanItems) {
        auto fetch = [&](int e, double& v1, double& v0, double& v2) {
            v1 = x1[r0 + e];
            if (HAS0) v0 = x0[r0 + e];
            if (HAS2) v2 = x2[r0 + e];
        };
        scan_round<HAS0, HAS2>(min(kFinThreads * kScanItems, pad - r0), (long long)b.n + r0, fetch,
                               x1, s1, x0, s0, x2, s2, s_w, st);
    }
}

}  // namespace

int bucket_count_for(int n) {
    int nbk = 1;
    while (nbk < kMaxBuckets && (n + nbk - 1) / nbk > kBucketTarget) nbk <<= 1;
    return nbk;
}

void launch_bucket_sort(const BucketArgs& b, bool has0, bool has2, bool sort_only, cudaStream_t st) {
    const size_t sm = 2ull * kBucketCap * sizeof(u64) + (2ull * kSub + 1) * sizeof(u32);
    static bool set = false;
    if (!set) {
        cudaFuncSetAttribute(k_bucket_finish<false, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
        cudaFuncSetAttribute(k_bucket_finish<true, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
        cudaFuncSetAttribute(k_bucket_finish<true, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
        cudaFuncSetAttribute(k_bucket_finish<false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
        set = true;
    }
    cudaMemsetAsync(b.hist, 0, (size_t)b.tile * b.nbk * sizeof(u32), st);
    cudaMemsetAsync(b.fallback, 0, sizeof(int), st);
    const dim3 grid((b.n + kCountThreads * kCountItems - 1) / (kCountThreads * kCountItems), b.tile);
    k_bucket_count<<<grid, kCountThreads, 0, st>>>(b);
    k_bucket_scan<<<(b.tile * 32 + 255) / 256, 256, 0, st>>>(b);
    k_bucket_scatter<<<grid, kCountThreads, 0, st>>>(b);
    if (sort_only) k_bucket_finish<false, false, true><<<b.tile, kFinThreads, sm, st>>>(b);
    else if (has2) k_bucket_finish<true, true, false><<<b.tile, kFinThreads, sm, st>>>(b);
    else if (has0) k_bucket_finish<true, false, false><<<b.tile, kFinThreads, sm, st>>>(b);
    else k_bucket_finish<false, false, false><<<b.tile, kFinThreads, sm, st>>>(b);
}

}  // namespace gtls
