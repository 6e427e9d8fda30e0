// Steps a1 (fold -> sortable keys, Eq. 10) and a2 (per-period stable phase sort,
// PAPER.md:185, ties by original index): general tiled path.
//
// A key packs floor(phase * 2^32) in the high word and the point index in the low word, so a
// stable LSD radix sort over the high word alone yields the order (key32, index).  Equal-key32
// runs (expected ~n^2 / 2^33 pairs per period) are then re-ordered by the full fp64 phase,
// which makes the permutation identical to a stable sort by fp64 phase.
#include "gtls_internal.cuh"

namespace gtls {

namespace {

__global__ void __launch_bounds__(256) k_fold_keys(TileArgs a, double* __restrict__ phase_out) {
    if (a.run_if && !*a.run_if) return;
    const long long total = (long long)a.tile * a.n;
    for (long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x; g < total;
         g += (long long)gridDim.x * blockDim.x) {
        const int pl = (int)(g / a.n), i = (int)(g - (long long)pl * a.n);
        const double ph = fold_phase(a.t[i], a.periods[a.p0 + pl]);
        a.keys_a[g] = ((u64)phase_key32(ph) << 32) | (u64)(u32)i;
        if (phase_out) phase_out[g] = ph;
    }
}

// ---- LSD radix pass: per-tile digit histogram ------------------------------------------
__global__ void __launch_bounds__(kRadixThreads) k_radix_hist(const u64* __restrict__ in,
                                                              u32* __restrict__ counts, int n,
                                                              int nt, int shift, const int* run_if) {
    __shared__ u32 h[256];
    if (run_if && !*run_if) return;
    const int tile = blockIdx.x, seg = blockIdx.y;
    h[threadIdx.x] = 0;
    __syncthreads();
    const u64* src = in + (long long)seg * n;
#pragma unroll
    for (int e = 0; e < kRadixItems; ++e) {
        const int i = tile * kRadixTile + e * kRadixThreads + threadIdx.x;
        if (i < n) atomicAdd(&h[(u32)(src[i] >> shift) & 255u], 1u);
    }
    __syncthreads();
    counts[((long long)seg * 256 + threadIdx.x) * nt + tile] = h[threadIdx.x];
}

// ---- exclusive scan over (digit-major, tile-minor) counts of one segment ------------------
__global__ void __launch_bounds__(256) k_radix_scan(u32* __restrict__ counts, int nt, const int* run_if) {
    if (run_if && !*run_if) return;
    __shared__ u32 s_tot[256];
    const int seg = blockIdx.x, d = threadIdx.x;
    u32* row = counts + ((long long)seg * 256 + d) * nt;
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
}

// ---- stable scatter ------------------------------------------------------------------------
// Warp w owns the contiguous sub-chunk [w*256, (w+1)*256) of the tile and walks it 32 keys at
// a time; __match_any_sync groups equal digits so each distinct digit costs one shared-memory
// counter update per round.  Order inside the tile = (warp, round, lane) = input order.
__global__ void __launch_bounds__(kRadixThreads) k_radix_scatter(const u64* __restrict__ in,
                                                                 u64* __restrict__ out,
                                                                 const u32* __restrict__ counts,
                                                                 int n, int nt, int shift, const int* run_if) {
    __shared__ u32 whist[kRadixWarps][256];
    if (run_if && !*run_if) return;
    const int tile = blockIdx.x, seg = blockIdx.y;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int k = threadIdx.x; k < kRadixWarps * 256; k += kRadixThreads) (&whist[0][0])[k] = 0;
    __syncthreads();
    const u64* src = in + (long long)seg * n;
    u64 key[kRadixItems];
    u32 lrank[kRadixItems];
#pragma unroll
    for (int r = 0; r < kRadixItems; ++r) {
        const int i = tile * kRadixTile + warp * (32 * kRadixItems) + r * 32 + lane;
        const bool valid = i < n;
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
        u32 acc = counts[((long long)seg * 256 + d) * nt + tile];
#pragma unroll
        for (int w = 0; w < kRadixWarps; ++w) { const u32 c = whist[w][d]; whist[w][d] = acc; acc += c; }
    }
    __syncthreads();
    u64* dst = out + (long long)seg * n;
#pragma unroll
    for (int r = 0; r < kRadixItems; ++r) {
        const int i = tile * kRadixTile + warp * (32 * kRadixItems) + r * 32 + lane;
        if (i < n) {
            const u32 d = (u32)(key[r] >> shift) & 255u;
            dst[whist[warp][d] + lrank[r]] = key[r];
        }
    }
}

// ---- tie fix-up: order equal-key32 runs by the full fp64 phase (stable) ---------------------
__global__ void __launch_bounds__(256) k_tie_fixup(TileArgs a, u64* __restrict__ keys) {
    if (a.run_if && !*a.run_if) return;
    const long long total = (long long)a.tile * a.n;
    for (long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x; g < total;
         g += (long long)gridDim.x * blockDim.x) {
        const int pl = (int)(g / a.n), s = (int)(g - (long long)pl * a.n);
        u64* seg = keys + (long long)pl * a.n;
        const u32 hi = (u32)(seg[s] >> 32);
        if (s + 1 >= a.n || (u32)(seg[s + 1] >> 32) != hi) continue;   // no run continues here
        if (s > 0 && (u32)(seg[s - 1] >> 32) == hi) continue;          // not the run's first key
        int e = s + 2;
        while (e < a.n && (u32)(seg[e] >> 32) == hi) ++e;
        const double period = a.periods[a.p0 + pl];
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

__global__ void __launch_bounds__(256) k_perm_export(const u64* __restrict__ keys, long long count,
                                                     int32_t* __restrict__ perm, const int* run_if) {
    if (run_if && !*run_if) return;
    for (long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x; g < count;
         g += (long long)gridDim.x * blockDim.x)
        perm[g] = (int32_t)(u32)keys[g];
}

inline int grid_for(long long total, int threads, int per_thread = 4) {
    long long b = (total + (long long)threads * per_thread - 1) / ((long long)threads * per_thread);
    if (b < 1) b = 1;
    if (b > 148LL * 32) b = 148LL * 32;
    return (int)b;
}

}  // namespace

void launch_fold_keys(const TileArgs& a, double* phase_out, cudaStream_t st) {
    k_fold_keys<<<grid_for((long long)a.tile * a.n, 256), 256, 0, st>>>(a, phase_out);
}

u64* launch_phase_sort(const TileArgs& a, cudaStream_t st, int* n_launches) {
    const int nt = (a.n + kRadixTile - 1) / kRadixTile;
    u64* src = a.keys_a;
    u64* dst = a.keys_b;
    const dim3 grid(nt, a.tile);
    for (int pass = 0; pass < 4; ++pass) {
        const int shift = 32 + 8 * pass;
        k_radix_hist<<<grid, kRadixThreads, 0, st>>>(src, a.counts, a.n, nt, shift, a.run_if);
        k_radix_scan<<<a.tile, 256, 0, st>>>(a.counts, nt, a.run_if);
        k_radix_scatter<<<grid, kRadixThreads, 0, st>>>(src, dst, a.counts, a.n, nt, shift, a.run_if);
        u64* tmp = src; src = dst; dst = tmp;
    }
    k_tie_fixup<<<grid_for((long long)a.tile * a.n, 256), 256, 0, st>>>(a, src);
    if (n_launches) *n_launches += 13;
    return src;   // after 4 passes the sorted keys are back in keys_a
}

void launch_perm_export(const u64* sorted, long long count, int32_t* out_perm, const int* run_if, cudaStream_t st) {
    k_perm_export<<<grid_for(count, 256), 256, 0, st>>>(sorted, count, out_perm, run_if);
}

}  // namespace gtls
