// Steps a1 (fold -> sortable keys, Eq. 10) and a2 (per-period stable phase sort,
// PAPER.md:185, ties by original index): LSD radix path.  It takes any phase distribution and is the
// fallback of the bucket fast path (bucket_sort.cu) for periods whose phases cluster; with
// a.seg_list == nullptr it processes every period of the tile (GTLS_SORT=lsd, A-B runs).
//
// A key packs floor(phase * 2^32) in the high word and the point index in the low word, so a
// stable LSD radix sort over the high word alone yields the order (key32, index).  Equal-key32
// runs (expected ~n^2 / 2^33 pairs per period) are then re-ordered by the full fp64 phase,
// which makes the permutation identical to a stable sort by fp64 phase.
#include "gtls_internal.cuh"

namespace gtls {

namespace {

// grid (chunks of n, segments): blockIdx.y strides over the segment list
__global__ void __launch_bounds__(256) k_fold_keys(TileArgs a, double* __restrict__ phase_out) {
    const int nseg = seg_count(a.seg_list, a.seg_count, a.tile);
    for (int s = blockIdx.y; s < nseg; s += gridDim.y) {
        const int pl = seg_at(a.seg_list, s);
        const double period = a.periods[a.p0 + pl];
        for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < a.n; i += gridDim.x * blockDim.x) {
            const double ph = fold_phase(a.t[i], period);
            const long long g = (long long)pl * a.n + i;
            a.keys_a[g] = ((u64)phase_key32(ph) << 32) | (u64)(u32)i;
            if (phase_out) phase_out[g] = ph;
        }
    }
}

// ---- LSD radix pass: per-chunk digit histogram ------------------------------------------
__global__ void __launch_bounds__(kRadixThreads) k_radix_hist(TileArgs a, const u64* __restrict__ in,
                                                              int nt, int shift) {
    __shared__ u32 h[256];
    const int chunk = blockIdx.x;
    const int nseg = seg_count(a.seg_list, a.seg_count, a.tile);
    for (int s = blockIdx.y; s < nseg; s += gridDim.y) {
        const int seg = seg_at(a.seg_list, s);
        h[threadIdx.x] = 0;
        __syncthreads();
        const u64* src = in + (long long)seg * a.n;
#pragma unroll
        for (int e = 0; e < kRadixItems; ++e) {
            const int i = chunk * kRadixTile + e * kRadixThreads + threadIdx.x;
            if (i < a.n) atomicAdd(&h[(u32)(src[i] >> shift) & 255u], 1u);
        }
        __syncthreads();
        a.counts[((long long)seg * 256 + threadIdx.x) * nt + chunk] = h[threadIdx.x];
        __syncthreads();
    }
}

// ---- exclusive scan over (digit-major, chunk-minor) counts of one segment ------------------
__global__ void __launch_bounds__(256) k_radix_scan(TileArgs a, int nt) {
    __shared__ u32 s_tot[256];
    const int d = threadIdx.x;
    const int nseg = seg_count(a.seg_list, a.seg_count, a.tile);
    for (int s = blockIdx.x; s < nseg; s += gridDim.x) {
        const int seg = seg_at(a.seg_list, s);
        u32* row = a.counts + ((long long)seg * 256 + d) * nt;
        u32 sum = 0;
        for (int k = 0; k < nt; ++k) sum += row[k];
        s_tot[d] = sum;
        __syncthreads();
        // exclusive scan of the 256 digit totals (Hillis-Steele in shared memory)
        u32 v = sum;
        for (int o = 1; o < 256; o <<= 1) {
            const u32 add = d >= o ? s_tot[d - o] : 0u;
            __syncthreads();
            v += add;
            s_tot[d] = v;
            __syncthreads();
        }
        u32 base = v - sum;
        for (int k = 0; k < nt; ++k) { const u32 c = row[k]; row[k] = base; base += c; }
        __syncthreads();
    }
}

// ---- stable scatter ------------------------------------------------------------------------
// Warp w owns the contiguous sub-chunk [w*256, (w+1)*256) of the chunk and walks it 32 keys at
// a time; __match_any_sync groups equal digits so each distinct digit costs one shared-memory
// counter update per round.  Order inside the chunk = (warp, round, lane) = input order.
__global__ void __launch_bounds__(kRadixThreads) k_radix_scatter(TileArgs a, const u64* __restrict__ in,
                                                                 u64* __restrict__ out, int nt, int shift) {
    __shared__ u32 whist[kRadixWarps][256];
    const int chunk = blockIdx.x;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nseg = seg_count(a.seg_list, a.seg_count, a.tile);
    for (int s = blockIdx.y; s < nseg; s += gridDim.y) {
        const int seg = seg_at(a.seg_list, s);
        for (int k = threadIdx.x; k < kRadixWarps * 256; k += kRadixThreads) (&whist[0][0])[k] = 0;
        __syncthreads();
        const u64* src = in + (long long)seg * a.n;
        u64 key[kRadixItems];
        u32 lrank[kRadixItems];
#pragma unroll
        for (int r = 0; r < kRadixItems; ++r) {
            const int i = chunk * kRadixTile + warp * (32 * kRadixItems) + r * 32 + lane;
            const bool valid = i < a.n;
            key[r] = valid ? src[i] : 0ull;
            const u32 d = valid ? ((u32)(key[r] >> shift) & 255u) : 256u;
            const u32 peers = __match_any_sync(0xffffffffu, d);
            const int leader = __ffs(peers) - 1;
            const u32 rank = __popc(peers & ((1u << lane) - 1u));
            u32 old = 0;
            if (valid && lane == leader) {
                old = whist[warp][d];
                whist[warp][d] = old + __popc(peers);
            }
            old = __shfl_sync(0xffffffffu, old, leader);
            lrank[r] = old + rank;
            __syncwarp();
        }
        __syncthreads();
        {   // digit d = threadIdx.x: exclusive prefix over warps, seeded with the global base
            const int d = threadIdx.x;
            u32 acc = a.counts[((long long)seg * 256 + d) * nt + chunk];
#pragma unroll
            for (int w = 0; w < kRadixWarps; ++w) { const u32 c = whist[w][d]; whist[w][d] = acc; acc += c; }
        }
        __syncthreads();
        u64* dst = out + (long long)seg * a.n;
#pragma unroll
        for (int r = 0; r < kRadixItems; ++r) {
            const int i = chunk * kRadixTile + warp * (32 * kRadixItems) + r * 32 + lane;
            if (i < a.n) {
                const u32 d = (u32)(key[r] >> shift) & 255u;
                dst[whist[warp][d] + lrank[r]] = key[r];
            }
        }
        __syncthreads();
    }
}

// ---- tie fix-up: order equal-key32 runs by the full fp64 phase (stable) ---------------------
__global__ void __launch_bounds__(256) k_tie_fixup(TileArgs a, u64* __restrict__ keys) {
    const int nseg = seg_count(a.seg_list, a.seg_count, a.tile);
    for (int sg = blockIdx.y; sg < nseg; sg += gridDim.y) {
        const int pl = seg_at(a.seg_list, sg);
        u64* seg = keys + (long long)pl * a.n;
        const double period = a.periods[a.p0 + pl];
        for (int s = blockIdx.x * blockDim.x + threadIdx.x; s < a.n; s += gridDim.x * blockDim.x) {
            const u32 hi = (u32)(seg[s] >> 32);
            if (s + 1 >= a.n || (u32)(seg[s + 1] >> 32) != hi) continue;   // no run continues here
            if (s > 0 && (u32)(seg[s - 1] >> 32) == hi) continue;          // not the run's first key
            int e = s + 2;
            while (e < a.n && (u32)(seg[e] >> 32) == hi) ++e;
            // stable insertion sort of seg[s..e) by phase; the run is already in index order
            for (int k = s + 1; k < e; ++k) {
                const u64 kk = seg[k];
                const double pk = fold_phase(a.t[(u32)kk], period);
                int m = k - 1;
                while (m >= s && fold_phase(a.t[(u32)seg[m]], period) > pk) { seg[m + 1] = seg[m]; --m; }
                seg[m + 1] = kk;
            }
        }
    }
}

__global__ void __launch_bounds__(256) k_perm_export(TileArgs a, const u64* __restrict__ keys,
                                                     int32_t* __restrict__ perm) {
    const int nseg = seg_count(a.seg_list, a.seg_count, a.tile);
    for (int sg = blockIdx.y; sg < nseg; sg += gridDim.y) {
        const long long base = (long long)seg_at(a.seg_list, sg) * a.n;
        for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < a.n; i += gridDim.x * blockDim.x)
            perm[base + i] = (int32_t)(u32)keys[base + i];
    }
}

// segments axis of the grid: every period of the tile, or a few CTAs striding over the fallback list
inline unsigned seg_grid(const TileArgs& a) { return a.seg_list ? (a.tile < 16 ? a.tile : 16) : a.tile; }
inline unsigned chunk_grid(int n, int per_cta) { const int b = (n + per_cta - 1) / per_cta; return b < 1 ? 1 : b; }

}  // namespace

void launch_fold_keys(const TileArgs& a, double* phase_out, cudaStream_t st) {
    k_fold_keys<<<dim3(chunk_grid(a.n, 1024), seg_grid(a)), 256, 0, st>>>(a, phase_out);
}

u64* launch_phase_sort(const TileArgs& a, cudaStream_t st, int* n_launches) {
    const int nt = (a.n + kRadixTile - 1) / kRadixTile;
    u64* src = a.keys_a;
    u64* dst = a.keys_b;
    const dim3 grid(nt, seg_grid(a));
    for (int pass = 0; pass < 4; ++pass) {
        const int shift = 32 + 8 * pass;
        k_radix_hist<<<grid, kRadixThreads, 0, st>>>(a, src, nt, shift);
        k_radix_scan<<<seg_grid(a), 256, 0, st>>>(a, nt);
        k_radix_scatter<<<grid, kRadixThreads, 0, st>>>(a, src, dst, nt, shift);
        u64* tmp = src; src = dst; dst = tmp;
    }
    k_tie_fixup<<<dim3(chunk_grid(a.n, 1024), seg_grid(a)), 256, 0, st>>>(a, src);
    if (n_launches) *n_launches += 13;
    return src;   // after 4 passes the sorted keys are back in keys_a
}

void launch_perm_export(const TileArgs& a, const u64* sorted, int32_t* out_perm, cudaStream_t st) {
    k_perm_export<<<dim3(chunk_grid(a.n, 1024), seg_grid(a)), 256, 0, st>>>(a, sorted, out_perm);
}

}  // namespace gtls
