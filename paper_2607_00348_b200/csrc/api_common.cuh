// Host-side helpers shared by the translation units of the C ABI (api_*.cu): error plumbing, the device
// block pool, the bump allocator over one device block, input staging, option defaults and the per-tile
// workspace geometry.  Not part of the ABI.
#pragma once
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <cmath>
#include <mutex>
#include <new>

#include "gtls_internal.cuh"

namespace gtls {
namespace api {

char* cuda_err_buf();                       // thread-local text of the last CUDA error (512 bytes)
int cuda_fail(cudaError_t e, const char* what);
#define CU(call)                                                          \
    do {                                                                  \
        cudaError_t e_ = (call);                                          \
        if (e_ != cudaSuccess) return ::gtls::api::cuda_fail(e_, #call);  \
    } while (0)

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

// Device blocks the library allocated itself are kept in a small pool between calls (api_pool.cu).
char* pool_take(size_t bytes, size_t* got);
void pool_give(char* base, size_t size);
size_t pool_cap();
void pool_release_all();

// Bump allocator over one device block.
struct Arena {
    char* base = nullptr;
    size_t size = 0, off = 0;
    bool owned = false;
    bool idle = false;      // set by the owner after its last stream synchronisation: nothing uses the block any more
    template <typename T>
    T* take(size_t count) {
        off = align_up(off);
        T* p = reinterpret_cast<T*>(base + off);
        off += count * sizeof(T);
        return off <= size ? p : nullptr;
    }
    ~Arena() {
        if (!owned || !base) return;
        if (!idle) cudaDeviceSynchronize();   // early returns: kernels of this call may still be running
        pool_give(base, size);
    }
};
int alloc_arena(Arena& ar, size_t bytes);

// Copies (host mode) or aliases (device mode) an input array.
template <typename T>
int stage_in(const T* src, size_t count, bool on_device, Arena& ar, cudaStream_t st, const T** out) {
    if (on_device) { *out = src; return GTLS_OK; }
    T* d = ar.take<T>(count);
    if (!d) return GTLS_ENOMEM;
    CU(cudaMemcpyAsync(d, src, count * sizeof(T), cudaMemcpyHostToDevice, st));
    *out = d;
    return GTLS_OK;
}

gtls_opts resolve_opts(const gtls_opts* in);

struct Timer {       // optional per-stage CUDA-event timing (opts->stats); owns its events
    bool on = false;
    cudaStream_t st = nullptr;
    cudaEvent_t ev[11] = {};
    void init(bool enable, cudaStream_t s) {
        on = enable; st = s;
        if (on) for (auto& e : ev) cudaEventCreate(&e);
    }
    void mark(int k) { if (on) cudaEventRecord(ev[k], st); }
    double ms(int a, int b) { float f = 0.f; cudaEventElapsedTime(&f, ev[a], ev[b]); return f; }
    ~Timer() { if (on) for (auto& e : ev) cudaEventDestroy(e); }
};


// ---- per-tile workspace geometry --------------------------------------------------------------------
struct Sizes {
    size_t fixed;        // per-call arrays
    size_t per_period;   // per period in flight
};

// pitch of the padded folded arrays for a largest duration fraction q_max
inline int pitch_for(long long n, double q_max) {
    long long dmax = (long long)(q_max * (double)n);
    if (dmax < 1) dmax = 1;
    if (dmax > n - 1) dmax = n - 1;
    return (int)((n + dmax + 7) / 8 * 8);
}

// per-period bytes of the bucket sort's scratch (16-bit CTA histograms, bucket starts, CTA offsets, flags)
inline size_t sort_scratch_bytes(long long n) {
    const size_t nbk = (size_t)bucket_count_for((int)n), ncta = (size_t)bucket_cta_count((int)n);
    return ncta * nbk * (sizeof(unsigned short) + sizeof(u32)) + (nbk + 3) * sizeof(u32) + 64;
}

inline Sizes workspace_sizes(long long n, long long n_per, int n_dur, double q_max, bool uniform) {
    Sizes s;
    const int pitch = pitch_for(n, q_max);
    const int spitch = pitch + 8;
    const int nt = (int)((n + kRadixTile - 1) / kRadixTile);
    s.fixed = 3 * align_up(n * sizeof(double)) + align_up(sizeof(CurveInfo)) +
              align_up(sizeof(SdeScratch)) + align_up(2 * sizeof(unsigned long long)) +
              2 * align_up(n_per * sizeof(double)) + align_up(n_per * sizeof(gtls_best)) + 4096 +
              align_up((size_t)kChi2Variants * (2 + kBinBlocks) * sizeof(int)) +
              align_up(2 * (size_t)(pitch - n + 2) * sizeof(double)) +      // gtab: D <= pitch - n
              2 * align_up(kXMargin * sizeof(double));
    s.per_period = 2 * n * sizeof(u64) + 256ull * nt * sizeof(u32) + n_dur * sizeof(DurEntry) +
                   n_dur * sizeof(Partial) + (size_t)kChi2Variants * n_dur * sizeof(int) +
                   n * sizeof(u32) + sort_scratch_bytes(n) +
                   (uniform ? 1 : 2) * ((size_t)pitch + spitch) * sizeof(double);
    return s;
}

#ifndef GTLS_FIN_SLOTS
#define GTLS_FIN_SLOTS (148 * 4)
#endif
constexpr long long kFinishSlots = GTLS_FIN_SLOTS;

inline int auto_tile(long long n_per, const Sizes& s, size_t budget) {
    long long t = (long long)(budget / s.per_period);
    if (t > 8192) t = 8192;
    // k_bucket_prefix and k_pad_scan run one CTA per period, 2 - 4 per SM at a time: a tile that is a multiple of
    // kFinishSlots (148 SMs x 4) leaves no partly filled last round
    if (t >= kFinishSlots && t < n_per) t -= t % kFinishSlots;
    if (t > n_per) t = n_per;
    if (t < 1) t = 1;
    return (int)t;
}

constexpr size_t kDefaultTileBudget = 24ull << 30;  // bytes of per-tile scratch when automatic


struct SortScratch { unsigned short* hist; u32* start; u32* rel; int* fb_flag; int* fb_list; int* fb_count; };
bool take_sort_scratch(Arena& ar, size_t tile, int n, SortScratch& sc);
// Steps a1-a4 for the tile described by `a` (api_search.cu)
void run_fold_sort_scan(TileArgs& a, const SortScratch& sc, double* x2, double* s2, int pad_override,
                        bool sort_only, double* phase_out, cudaStream_t st, int* launches);

}  // namespace api
}  // namespace gtls
