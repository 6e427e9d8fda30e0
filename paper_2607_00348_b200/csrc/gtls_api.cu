// C ABI of libgtls (include/gtls.h): argument validation, device memory, the period-tile
// loop and the epilogue.  All arithmetic of the search runs in the kernels of pre.cu,
// fold_sort.cu, scan.cu, chi2.cu and epilogue.cu; there is no CPU fallback.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <cmath>
#include <mutex>
#include <new>
#include <thread>
#include <vector>

#include "gtls_internal.cuh"

using namespace gtls;

namespace {

thread_local char g_cuda_err[512] = "";

int cuda_fail(cudaError_t e, const char* what) {
    snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s (%s)", what, cudaGetErrorString(e),
             cudaGetErrorName(e));
    return GTLS_ECUDA;
}
#define CU(call)                                                   \
    do {                                                           \
        cudaError_t e_ = (call);                                   \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call);        \
    } while (0)

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

// Device blocks the library allocated itself are kept in a small pool between calls (cudaMalloc and
// cudaFree of a few GB cost milliseconds each and cudaFree synchronises the device: half of the end-to-end
// time of a short light curve through host buffers).  At most kPoolSlots free blocks, each at most
// GTLS_CACHE_MB (default 8192) MiB; gtls_release_cache() frees them; GTLS_CACHE_MB=0 switches the pool off.
constexpr int kPoolSlots = 4;
struct PoolBlock { char* base; size_t size; int dev; };
std::mutex g_pool_mu;
PoolBlock g_pool[kPoolSlots] = {};
size_t pool_cap() {
    static const size_t cap = [] { const char* e = getenv("GTLS_CACHE_MB"); return (size_t)(e ? atoll(e) : 8192) << 20; }();
    return cap;
}
char* pool_take(size_t bytes, size_t* got) {
    int dev = -1;
    if (pool_cap() == 0 || cudaGetDevice(&dev) != cudaSuccess) return nullptr;
    std::lock_guard<std::mutex> lk(g_pool_mu);
    int best = -1;
    for (int i = 0; i < kPoolSlots; ++i)
        if (g_pool[i].base && g_pool[i].dev == dev && g_pool[i].size >= bytes &&
            (best < 0 || g_pool[i].size < g_pool[best].size)) best = i;
    if (best < 0) return nullptr;
    char* p = g_pool[best].base; *got = g_pool[best].size;
    g_pool[best] = PoolBlock{};
    return p;
}
void pool_give(char* base, size_t size) {
    int dev = -1;
    if (size <= pool_cap() && cudaGetDevice(&dev) == cudaSuccess) {
        std::lock_guard<std::mutex> lk(g_pool_mu);
        int slot = -1;
        for (int i = 0; i < kPoolSlots; ++i) if (!g_pool[i].base) { slot = i; break; }
        if (slot < 0) {                       // full: the smallest block makes room if it is smaller than this one
            int sm = 0;
            for (int i = 1; i < kPoolSlots; ++i) if (g_pool[i].size < g_pool[sm].size) sm = i;
            if (g_pool[sm].size < size) { cudaFree(g_pool[sm].base); slot = sm; }
        }
        if (slot >= 0) { g_pool[slot] = PoolBlock{base, size, dev}; return; }
    }
    cudaFree(base);
}

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

Sizes workspace_sizes(long long n, long long n_per, int n_dur, double q_max, bool uniform) {
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
                   n * sizeof(u32) + (4ull * kMaxBuckets + 3) * sizeof(u32) + 3ull * kMaxBuckets * sizeof(double) +
                   (uniform ? 1 : 2) * ((size_t)pitch + spitch) * sizeof(double);
    return s;
}

#ifndef GTLS_FIN_SLOTS
#define GTLS_FIN_SLOTS (148 * 4)
#endif
constexpr long long kFinishSlots = GTLS_FIN_SLOTS;

int auto_tile(long long n_per, const Sizes& s, size_t budget) {
    long long t = (long long)(budget / s.per_period);
    if (t > 8192) t = 8192;
    // k_bucket_finish runs one CTA per period, kFinishSlots of them at a time (148 SMs x 5 CTAs): a tile
    // that is a multiple of that leaves no partly filled last round
    if (t >= kFinishSlots && t < n_per) t -= t % kFinishSlots;
    if (t > n_per) t = n_per;
    if (t < 1) t = 1;
    return (int)t;
}

constexpr size_t kDefaultTileBudget = 24ull << 30;  // bytes of per-tile scratch when automatic

gtls_opts resolve_opts(const gtls_opts* in) {
    gtls_opts o;
    gtls_opts_default(&o);
    if (in) {
        size_t sz = in->struct_size ? in->struct_size : sizeof(gtls_opts);
        if (sz > sizeof(gtls_opts)) sz = sizeof(gtls_opts);
        memcpy(&o, in, sz);
        o.struct_size = sizeof(gtls_opts);
    }
    return o;
}

struct Timer {       // optional per-stage CUDA-event timing (opts->stats)
    bool on = false;
    cudaStream_t st = nullptr;
    cudaEvent_t ev[9] = {};
    void init(bool enable, cudaStream_t s) {
        on = enable; st = s;
        if (on) for (auto& e : ev) cudaEventCreate(&e);
    }
    void mark(int k) { if (on) cudaEventRecord(ev[k], st); }
    double ms(int a, int b) { float f = 0.f; cudaEventElapsedTime(&f, ev[a], ev[b]); return f; }
    ~Timer() { if (on) for (auto& e : ev) cudaEventDestroy(e); }
};

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

int alloc_arena(Arena& ar, size_t bytes) {
    size_t got = 0;
    if (char* p = pool_take(bytes, &got)) { ar.base = p; ar.size = got; ar.off = 0; ar.owned = true; return GTLS_OK; }
    if (pool_cap() && bytes <= pool_cap()) bytes = align_up(bytes + bytes / 16, 2u << 20);   // slack: the next, slightly larger request fits too
    cudaError_t e = cudaMalloc((void**)&ar.base, bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        gtls_release_cache();                  // the pool may hold what this request needs
        e = cudaMalloc((void**)&ar.base, bytes);
    }
    if (e != cudaSuccess) { cudaGetLastError(); ar.base = nullptr; snprintf(g_cuda_err, sizeof(g_cuda_err), "cudaMalloc(%zu): %s", bytes, cudaGetErrorString(e)); return GTLS_ENOMEM; }
    ar.size = bytes; ar.off = 0; ar.owned = true;
    return GTLS_OK;
}

// Shared front end of the debug exports: curve arrays + sorted keys for `tile` periods.
struct CurveDev {
    const double *t = nullptr, *y = nullptr, *dy = nullptr;
    double *wr = nullptr, *w = nullptr, *wr2 = nullptr;
    CurveInfo* info = nullptr;
};


struct SortScratch { u32* hist; u32* start; u32* cursor; int* fb_flag; int* fb_list; int* fb_count; };

bool take_sort_scratch(Arena& ar, size_t tile, int nbk, SortScratch& sc) {
    sc.hist = ar.take<u32>(tile * nbk);
    sc.start = ar.take<u32>(tile * (nbk + 1));
    sc.cursor = ar.take<u32>(tile * nbk);
    sc.fb_flag = ar.take<int>(tile);
    sc.fb_list = ar.take<int>(tile);
    sc.fb_count = ar.take<int>(1);
    return sc.fb_count != nullptr;
}

bool force_lsd_sort() {
    static const bool f = [] { const char* e = getenv("GTLS_SORT"); return e && strcmp(e, "lsd") == 0; }();
    return f;
}

}  // namespace

SideStream* gtls::side_stream(int which) {
    struct Slot {
        SideStream ss{};
        bool ok = false;
        int dev = -1;
        Slot() {
            int lo = 0, hi = 0;
            if (cudaGetDevice(&dev) != cudaSuccess) return;
            if (cudaDeviceGetStreamPriorityRange(&lo, &hi) != cudaSuccess) return;
            if (cudaStreamCreateWithPriority(&ss.s, cudaStreamNonBlocking, hi) != cudaSuccess) return;
            if (cudaEventCreateWithFlags(&ss.fork, cudaEventDisableTiming) != cudaSuccess) return;
            if (cudaEventCreateWithFlags(&ss.join, cudaEventDisableTiming) != cudaSuccess) return;
            ok = true;
        }
        ~Slot() {     // worker threads of gtls_search_batch end after every call
            if (ss.s) cudaStreamDestroy(ss.s);
            if (ss.fork) cudaEventDestroy(ss.fork);
            if (ss.join) cudaEventDestroy(ss.join);
        }
    };
    static const bool enabled = [] { const char* e = getenv("GTLS_STREAMS"); return !(e && atoi(e) == 0); }();
    if (!enabled || which < 0 || which > 1) return nullptr;
    static thread_local Slot slots[2];
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return nullptr;
    Slot& sl = slots[which];
    return (sl.ok && sl.dev == dev) ? &sl.ss : nullptr;
}

namespace {

// Steps a1-a4 for the tile described by `a` (a.perm, a.x1/s1[/x0/s0] are outputs).
//   The bucket fast path first; a period with a bucket larger than kBucketCap (clustered phases) is put
//   on the tile's fallback list on the device and skipped by the fast path; the LSD radix path
//   (fold_sort.cu + scan.cu) then runs over that list (a handful of CTAs that find it empty, normally).
//   GTLS_SORT=lsd: the LSD path for every period (A-B runs, tests).
// sort_only: permutation only.  phase_out: also export the phases (Eq. 10).
void run_fold_sort_scan(TileArgs& a, const SortScratch& sc, double* x2, double* s2, int pad_override,
                        bool sort_only, double* phase_out, cudaStream_t st, int* launches) {
    a.seg_list = nullptr; a.seg_count = nullptr;
    int nl = 0;
    if (!force_lsd_sort()) {
        BucketArgs b;
        memset(&b, 0, sizeof(b));
        b.n = a.n; b.tile = a.tile; b.p0 = a.p0; b.n_dur = a.n_dur; b.pad_override = pad_override;
        b.nbk = bucket_count_for(a.n);
        int lg = 0; while ((1 << lg) < b.nbk) ++lg;
        b.shift = 32 - lg;
        b.pitch = a.pitch; b.spitch = a.spitch;
        b.t = a.t; b.wr = a.wr; b.w = a.w; b.wr2 = a.wr2; b.periods = a.periods; b.durtab = a.durtab;
        b.hist = sc.hist; b.start = sc.start; b.cursor = sc.cursor;
        b.fb_flag = sc.fb_flag; b.fb_list = sc.fb_list; b.fb_count = sc.fb_count;
        b.keys = a.keys_b; b.perm = a.perm;
        b.x1 = a.x1; b.s1 = a.s1; b.x0 = a.x0; b.s0 = a.s0; b.x2 = x2; b.s2 = s2;
        const bool has2 = s2 != nullptr, has0 = !a.uniform || has2;
        launch_bucket_sort_head(b, st);
        // the fallback list is known: the LSD path over it (a handful of CTAs, a few hundred microseconds
        // of latency when a period is on the list) runs beside the fast path on a side stream
        cudaStream_t ls = st;
        SideStream* side = side_stream(1);
        if (side) {
            cudaEventRecord(side->fork, st);
            cudaStreamWaitEvent(side->s, side->fork, 0);
            ls = side->s;
        }
        launch_bucket_sort_tail(b, has0, has2, sort_only, st);
        nl += sort_only ? 4 : 5;
        a.seg_list = sc.fb_list; a.seg_count = sc.fb_count;
        launch_fold_keys(a, nullptr, ls);
        int l2 = 0;
        const u64* sorted = launch_phase_sort(a, ls, &l2);
        if (!sort_only) launch_gather_scan(a, sorted, x2, s2, pad_override, ls);
        launch_perm_export(a, sorted, (int32_t*)a.perm, ls);
        if (side) {
            cudaEventRecord(side->join, ls);
            cudaStreamWaitEvent(st, side->join, 0);
        }
        if (phase_out) {                          // phases of every period: the LSD path's fold kernel, dense
            a.seg_list = nullptr; a.seg_count = nullptr;
            launch_fold_keys(a, phase_out, st); ++nl;
        }
        a.seg_list = nullptr; a.seg_count = nullptr;
        if (launches) *launches += nl + 1 + l2 + (sort_only ? 0 : 1) + 1;
        return;
    }
    launch_fold_keys(a, phase_out, st);
    int l2 = 0;
    const u64* sorted = launch_phase_sort(a, st, &l2);
    if (!sort_only) launch_gather_scan(a, sorted, x2, s2, pad_override, st);
    launch_perm_export(a, sorted, (int32_t*)a.perm, st);
    if (launches) *launches += nl + 1 + l2 + (sort_only ? 0 : 1) + 1;
}

}  // namespace

extern "C" {

void gtls_opts_default(gtls_opts* o) {
    if (!o) return;
    memset(o, 0, sizeof(*o));
    o->struct_size = sizeof(gtls_opts);
    o->dt0 = 0.05;
    o->sde_kernel = 151;
}

const char* gtls_version(void) { return "gtls-b200 0.1.0 (sm_100a)"; }

void gtls_release_cache(void) {
    std::lock_guard<std::mutex> lk(g_pool_mu);
    for (auto& b : g_pool) { if (b.base) cudaFree(b.base); b = PoolBlock{}; }
}
const char* gtls_last_cuda_error(void) { return g_cuda_err; }

const char* gtls_strerror(int code) {
    switch (code) {
        case GTLS_OK: return "ok";
        case GTLS_EINVAL: return "invalid argument";
        case GTLS_ENONFINITE: return "non-finite value in t/y/dy, or dy <= 0";
        case GTLS_EGRID: return "period <= 0 or duration fraction outside (0, 0.5]";
        case GTLS_ENOMEM: return "out of device memory or workspace too small";
        case GTLS_ECUDA: return "CUDA error (see gtls_last_cuda_error)";
        case GTLS_EDEGENERATE: return "degenerate spectrum (chi2_min == 0 or sigma_SR == 0); SDE set to 0";
        case GTLS_EUNSUPPORTED: return "option not supported";
        default: return "unknown error code";
    }
}

size_t gtls_workspace_bytes(int64_t n, int64_t n_per, int32_t n_dur, const gtls_opts* opts) {
    if (n < 3 || n_per < 1 || n_dur < 1) return 0;
    const gtls_opts o = resolve_opts(opts);
    const Sizes s = workspace_sizes(n, n_per, n_dur, 0.5, false);     // worst case
    const int tile = o.period_tile > 0 ? (int)(o.period_tile < n_per ? o.period_tile : n_per)
                                       : auto_tile(n_per, s, kDefaultTileBudget);
    return s.fixed + (size_t)tile * align_up(s.per_period) + 64 * 256;
}

int gtls_search(const double* t, const double* y, const double* dy, int64_t n,
                const double* period_grid, int64_t n_per, const double* duration_grid,
                int32_t n_dur, const double* tmpl, int32_t n_tmpl, const gtls_opts* opts,
                double* out_chi2, gtls_best* out_best, double* out_sde_raw, double* out_sde,
                gtls_summary* out_summary) {
    g_cuda_err[0] = 0;
    const gtls_opts o = resolve_opts(opts);
    if (!t || !y || !dy || !period_grid || !duration_grid || !tmpl || !out_chi2) return GTLS_EINVAL;
    if (n < 3 || n > 0x3fffffff || n_per < 1 || n_dur < 1 || n_dur > 4096 || n_tmpl < 2) return GTLS_EINVAL;
    if (!(o.dt0 >= 0.0) || o.sde_kernel < 0 || (o.sde_kernel > 1 && o.sde_kernel % 2 == 0)) return GTLS_EINVAL;
    if (o.path < 0 || o.path > 2 || o.period_tile < 0) return GTLS_EINVAL;
    if (o.top_k < 0) return GTLS_EINVAL;
    if (o.top_k > kTopKMax || (o.top_k > 0 && o.chi2_fp32)) return GTLS_EUNSUPPORTED;
    if (o.chi2_fp32 != 0 && o.chi2_fp32 != 1) return GTLS_EINVAL;
    if (o.path == 1) return GTLS_EUNSUPPORTED;   // fused shared-memory path: not built yet
    CU(cudaSetDevice(o.device));
    cudaStream_t st = (cudaStream_t)o.stream;
    const bool dev = o.pointers_on_device != 0;
    const long long n_durs_total = o.dur_per_period ? n_per * (long long)n_dur : n_dur;

    // ---- device memory -----------------------------------------------------------------
    Arena io;          // host mode: staged inputs and outputs
    if (!dev) {
        size_t bytes = 3 * align_up(n * 8) + align_up(n_per * 8) + align_up(n_durs_total * 8) +
                       align_up(n_tmpl * 8) + 3 * align_up(n_per * 8) +
                       align_up(n_per * sizeof(gtls_best)) + 16 * 256;
        int rc = alloc_arena(io, bytes);
        if (rc) return rc;
    }
    const double *d_t, *d_y, *d_dy, *d_per, *d_dur, *d_tmpl;
    int rc;
    if ((rc = stage_in(t, n, dev, io, st, &d_t))) return rc;
    if ((rc = stage_in(y, n, dev, io, st, &d_y))) return rc;
    if ((rc = stage_in(dy, n, dev, io, st, &d_dy))) return rc;
    if ((rc = stage_in(period_grid, n_per, dev, io, st, &d_per))) return rc;
    if ((rc = stage_in(duration_grid, n_durs_total, dev, io, st, &d_dur))) return rc;
    if ((rc = stage_in(tmpl, n_tmpl, dev, io, st, &d_tmpl))) return rc;
    double* d_chi2 = dev ? out_chi2 : io.take<double>(n_per);
    double* d_sde_raw_out = dev ? out_sde_raw : (out_sde_raw ? io.take<double>(n_per) : nullptr);
    double* d_sde_out = dev ? out_sde : (out_sde ? io.take<double>(n_per) : nullptr);
    gtls_best* d_best_out = dev ? out_best : (out_best ? io.take<gtls_best>(n_per) : nullptr);
    if (!d_chi2) return GTLS_ENOMEM;

    Arena ws;
    const Sizes worst = workspace_sizes(n, n_per, n_dur, 0.5, false);
    if (o.workspace) {
        ws.base = (char*)o.workspace; ws.size = o.workspace_bytes; ws.owned = false;
        if (((uintptr_t)ws.base & 255) != 0) return GTLS_EINVAL;
        if (ws.size < worst.fixed + align_up(worst.per_period)) return GTLS_ENOMEM;
    } else {
        // own scratch: the automatic tile, shrunk so that it takes at most half of the free device memory
        size_t need = gtls_workspace_bytes(n, n_per, n_dur, &o);
        size_t free_b = 0, total_b = 0;
        if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess && need > free_b / 2) {
            const size_t floor_b = worst.fixed + align_up(worst.per_period) + 64 * 256;
            need = free_b / 2 > floor_b ? free_b / 2 : floor_b;
        }
        if ((rc = alloc_arena(ws, need))) return rc;
    }
    double* d_wr = ws.take<double>(n);
    double* d_w = ws.take<double>(n);
    double* d_wr2 = ws.take<double>(n);
    CurveInfo* d_info = ws.take<CurveInfo>(1);
    SdeScratch* d_sde_sc = ws.take<SdeScratch>(1);
    unsigned long long* d_counters = ws.take<unsigned long long>(2);
    double* d_sde_raw = d_sde_raw_out ? d_sde_raw_out : ws.take<double>(n_per);
    double* d_sde = d_sde_out ? d_sde_out : ws.take<double>(n_per);
    gtls_best* d_best = d_best_out ? d_best_out : ws.take<gtls_best>(n_per);
    if (!d_best) return GTLS_ENOMEM;

    Timer tm;
    tm.init(o.stats != nullptr, st);
    cudaEvent_t ev_begin = nullptr, ev_end = nullptr;
    if (o.stats) { cudaEventCreate(&ev_begin); cudaEventCreate(&ev_end); cudaEventRecord(ev_begin, st); }
    gtls_stats stats;
    memset(&stats, 0, sizeof(stats));

    // ---- a0: per-curve arrays + validation ----------------------------------------------
    tm.mark(0);
    CU(cudaMemsetAsync(d_info, 0, sizeof(CurveInfo), st));
    CU(cudaMemsetAsync(d_counters, 0, 2 * sizeof(unsigned long long), st));
    launch_curve_pre(d_t, d_y, d_dy, (int)n, d_wr, d_w, d_wr2, d_info, st);
    launch_grid_check(d_per, n_per, d_dur, n_durs_total, d_info, st);
    stats.kernel_launches += 2;
    CurveInfo info;
    CU(cudaMemcpyAsync(&info, d_info, sizeof(info), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    CU(cudaGetLastError());
    if (info.bad_curve) return GTLS_ENONFINITE;
    if (info.bad_period || info.bad_duration) return GTLS_EGRID;
    tm.mark(1);
    if (o.stats) { CU(cudaStreamSynchronize(st)); stats.ms_pre += tm.ms(0, 1); }
    const bool uniform = info.w_min == info.w_max;

    const double* gtab_dev = nullptr;
    int gtab_max = 0;
    {   // template sums per D, once per search (every D the grid can ask for: D <= floor(q_max * n) <= pitch - n)
        long long dmax = (long long)(info.q_max * (double)n);
        dmax = dmax < 1 ? 1 : (dmax > n - 1 ? n - 1 : dmax);
        double* gtab = ws.take<double>(2 * (size_t)(dmax + 1));
        if (!gtab) return GTLS_ENOMEM;
        launch_gtab(d_tmpl, n_tmpl, (int)dmax, gtab, st);
        stats.kernel_launches += 1;
        gtab_dev = gtab; gtab_max = (int)dmax;
    }

    // ---- tile geometry -------------------------------------------------------------------
    const Sizes sz = workspace_sizes(n, n_per, n_dur, info.q_max, uniform);
    const size_t avail = ws.size - align_up(ws.off) - 32 * 256;
    long long tile_cap = (long long)(avail / align_up(sz.per_period + 8 * 256));
    int tile = o.period_tile > 0 ? o.period_tile : auto_tile(n_per, sz, kDefaultTileBudget);
    if (tile > tile_cap) tile = (int)tile_cap;
    if (o.period_tile <= 0 && tile >= kFinishSlots && tile < n_per) tile -= (int)(tile % kFinishSlots);   // see auto_tile
    if (tile > n_per) tile = (int)n_per;
    if (tile < 1) return GTLS_ENOMEM;
    TileArgs a;
    memset(&a, 0, sizeof(a));
    a.n = (int)n; a.n_dur = n_dur; a.n_tmpl = n_tmpl; a.dur_per_period = o.dur_per_period;
    a.dt0 = o.dt0; a.uniform = uniform ? 1 : 0; a.w_uniform = info.w_min; a.chi2_fp32 = o.chi2_fp32; a.top_k = o.top_k;
    a.pitch = pitch_for(n, info.q_max); a.spitch = a.pitch + 8;
    a.t = d_t; a.wr = d_wr; a.w = d_w; a.wr2 = d_wr2; a.periods = d_per; a.durs = d_dur;
    a.tmpl = d_tmpl; a.chi2_0 = &d_info->chi2_0;
    const int nt = (int)((n + kRadixTile - 1) / kRadixTile);
    a.keys_a = ws.take<u64>((size_t)tile * n);
    a.keys_b = ws.take<u64>((size_t)tile * n);
    a.counts = ws.take<u32>((size_t)tile * 256 * nt);
    a.perm = ws.take<u32>((size_t)tile * n);
    SortScratch ssc;
    if (!take_sort_scratch(ws, (size_t)tile, bucket_count_for((int)n), ssc)) return GTLS_ENOMEM;
    a.durtab = ws.take<DurEntry>((size_t)tile * n_dur);
    a.gtab = gtab_dev; a.gtab_max = gtab_max;
    a.partial = ws.take<Partial>((size_t)tile * n_dur);
    a.trial_list = ws.take<int>((size_t)kChi2Variants * tile * n_dur);
    a.trial_count = ws.take<int>((size_t)kChi2Variants * (2 + kBinBlocks));   // totals, the per-CTA counts of k_bin_trials, the trial queues
    a.x1 = ws.take<double>((size_t)tile * a.pitch + kXMargin);      // + the last period's zero margin
    a.s1 = ws.take<double>((size_t)tile * a.spitch);
    if (!uniform) {
        a.x0 = ws.take<double>((size_t)tile * a.pitch + kXMargin);
        a.s0 = ws.take<double>((size_t)tile * a.spitch);
    }
    if (!a.s1 || (!uniform && !a.s0)) return GTLS_ENOMEM;

    SdeScratch sc;
    unsigned long long counters[2];
    // ---- period tiles ----------------------------------------------------------------------
    for (long long p0 = 0; p0 < n_per; p0 += tile) {
        a.p0 = p0;
        a.tile = (int)((n_per - p0) < tile ? (n_per - p0) : tile);
        int launches = 0;
        tm.mark(0);
        launch_durtab(a, st);
        tm.mark(1);
        tm.mark(2);
        run_fold_sort_scan(a, ssc, nullptr, nullptr, -1, false, nullptr, st, &launches);
        tm.mark(3);
        tm.mark(4);
        if (a.top_k > 0) launch_chi2_topk(a, st);
        else launch_chi2_ring(a, st);
        tm.mark(5);
        launch_reduce(a, d_chi2, d_best, d_counters, st);
        tm.mark(6);
        stats.kernel_launches += launches + 2 + (a.top_k > 0 ? 1 : 2 + (uniform ? kChi2Variants - 1 : kChi2Variants - 3));   // k_bin_trials is two launches
        stats.chi2_launches += 1;
        if (o.stats) {
            CU(cudaStreamSynchronize(st));
            stats.ms_pre += tm.ms(0, 1); stats.ms_fold += tm.ms(1, 2); stats.ms_sort += tm.ms(2, 3);
            stats.ms_scan += tm.ms(3, 4); stats.ms_chi2 += tm.ms(4, 5); stats.ms_reduce += tm.ms(5, 6);
        }
    }
    CU(cudaGetLastError());

    // ---- a9: SR / SDE epilogue --------------------------------------------------------------
    tm.mark(0);
    int launches = 0;
    launch_sde(d_chi2, n_per, o.sde_kernel, d_sde_raw, d_sde, d_sde_sc, st, &launches);
    stats.kernel_launches += launches;
    tm.mark(1);
    CU(cudaMemcpyAsync(&sc, d_sde_sc, sizeof(sc), cudaMemcpyDeviceToHost, st));
    CU(cudaMemcpyAsync(counters, d_counters, sizeof(counters), cudaMemcpyDeviceToHost, st));
    if (o.stats) cudaEventRecord(ev_end, st);
    CU(cudaStreamSynchronize(st));
    CU(cudaGetLastError());
    if (o.stats) stats.ms_epilogue = tm.ms(0, 1);

    if (out_summary) {
        gtls_best b;
        double period = 0.0;
        CU(cudaMemcpyAsync(&b, d_best + sc.argmin, sizeof(b), cudaMemcpyDeviceToHost, st));
        CU(cudaMemcpyAsync(&period, d_per + sc.argmin, sizeof(double), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        out_summary->best_period_idx = sc.argmin;
        out_summary->best_dur_idx = b.dur_idx;
        out_summary->best_start = b.start;
        out_summary->best_period = period;
        out_summary->best_t0 = b.t0;
        out_summary->best_depth = b.depth;
        out_summary->chi2_min = sc.chi2_min;
        out_summary->chi2_null = info.chi2_0;
        out_summary->sde_raw_max = sc.sde_raw_best;
        out_summary->sde_max = sc.sde_max;
        out_summary->sde_argmax = sc.sde_argmax;
        out_summary->windows_evaluated = (int64_t)counters[0];
    }
    if (!dev) {
        CU(cudaMemcpyAsync(out_chi2, d_chi2, n_per * sizeof(double), cudaMemcpyDeviceToHost, st));
        if (out_best) CU(cudaMemcpyAsync(out_best, d_best, n_per * sizeof(gtls_best), cudaMemcpyDeviceToHost, st));
        if (out_sde_raw) CU(cudaMemcpyAsync(out_sde_raw, d_sde_raw, n_per * sizeof(double), cudaMemcpyDeviceToHost, st));
        if (out_sde) CU(cudaMemcpyAsync(out_sde, d_sde, n_per * sizeof(double), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
    }
    if (o.stats) {
        float f = 0.f;
        cudaEventElapsedTime(&f, ev_begin, ev_end);
        stats.ms_total = f;
        stats.windows = (int64_t)counters[0];
        stats.window_points = (int64_t)counters[1];
        stats.period_points = n * n_per;
        stats.period_tile = tile;
        stats.path = 2;
        stats.uniform_dy = uniform ? 1 : 0;
        *o.stats = stats;
        cudaEventDestroy(ev_begin); cudaEventDestroy(ev_end);
    }
    io.idle = ws.idle = true;                 // the stream was synchronised after the last use of both
    return sc.degenerate ? GTLS_EDEGENERATE : GTLS_OK;
}

int gtls_fold_sort(const double* t, int64_t n, const double* periods, int64_t n_per,
                   const gtls_opts* opts, double* out_phase, int32_t* out_perm) {
    g_cuda_err[0] = 0;
    const gtls_opts o = resolve_opts(opts);
    if (!t || !periods || !out_perm || n < 1 || n > 0x3fffffff || n_per < 1) return GTLS_EINVAL;
    CU(cudaSetDevice(o.device));
    cudaStream_t st = (cudaStream_t)o.stream;
    const bool dev = o.pointers_on_device != 0;
    const int nt = (int)((n + kRadixTile - 1) / kRadixTile);
    const int nbk = bucket_count_for((int)n);
    const size_t per_period = 2 * n * sizeof(u64) + 256ull * nt * sizeof(u32) + n * sizeof(u32) +
                              (4ull * nbk + 1) * sizeof(u32) + 3ull * nbk * sizeof(double) +
                              (dev ? 0 : n * (sizeof(double) + sizeof(int32_t))) + 1024;
    long long tile = (long long)((1ull << 30) / per_period);
    if (o.period_tile > 0) tile = o.period_tile;
    if (tile > n_per) tile = n_per;
    if (tile < 1) tile = 1;
    Arena ar;
    int rc = alloc_arena(ar, align_up(n * 8) + align_up(n_per * 8) + tile * align_up(per_period) + 32 * 256);
    if (rc) return rc;
    const double *d_t, *d_per;
    if ((rc = stage_in(t, n, dev, ar, st, &d_t))) return rc;
    if ((rc = stage_in(periods, n_per, dev, ar, st, &d_per))) return rc;
    TileArgs a;
    memset(&a, 0, sizeof(a));
    a.n = (int)n; a.t = d_t; a.periods = d_per;
    a.keys_a = ar.take<u64>((size_t)tile * n);
    a.keys_b = ar.take<u64>((size_t)tile * n);
    a.counts = ar.take<u32>((size_t)tile * 256 * nt);
    SortScratch ssc;
    if (!take_sort_scratch(ar, (size_t)tile, nbk, ssc)) return GTLS_ENOMEM;
    double* d_phase = dev ? nullptr : (out_phase ? ar.take<double>((size_t)tile * n) : nullptr);
    int32_t* d_perm = dev ? nullptr : ar.take<int32_t>((size_t)tile * n);
    if (!a.counts || (!dev && !d_perm)) return GTLS_ENOMEM;
    for (long long p0 = 0; p0 < n_per; p0 += tile) {
        a.p0 = p0;
        a.tile = (int)((n_per - p0) < tile ? (n_per - p0) : tile);
        const size_t cnt = (size_t)a.tile * n;
        double* ph = dev ? (out_phase ? out_phase + p0 * n : nullptr) : d_phase;
        int32_t* pm = dev ? out_perm + p0 * n : d_perm;
        a.perm = (u32*)pm;
        run_fold_sort_scan(a, ssc, nullptr, nullptr, 0, true, ph, st, nullptr);
        if (!dev) {
            if (out_phase) CU(cudaMemcpyAsync(out_phase + p0 * n, ph, cnt * sizeof(double), cudaMemcpyDeviceToHost, st));
            CU(cudaMemcpyAsync(out_perm + p0 * n, pm, cnt * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
            CU(cudaStreamSynchronize(st));
        }
    }
    CU(cudaStreamSynchronize(st));
    CU(cudaGetLastError());
    return GTLS_OK;
}

// Front end shared by the single-period debug exports: curve arrays, sorted keys, padded
// prefix sums of x1, x0, x2 for one period with `pad` wrap entries.
static int one_period_scan(const double* t, const double* y, const double* dy, int64_t n,
                           double period, int64_t pad, const gtls_opts& o, Arena& ar, TileArgs& a,
                           double** d_s2) {
    cudaStream_t st = (cudaStream_t)o.stream;
    const bool dev = o.pointers_on_device != 0;
    const int nt = (int)((n + kRadixTile - 1) / kRadixTile);
    const int pitch = (int)((n + pad + 7) / 8 * 8), spitch = pitch + 8;
    size_t bytes = 9 * align_up(n * 8) + 2 * align_up(n * sizeof(u64)) + align_up(256ull * nt * 4) + 32768 +
                   3 * align_up((size_t)pitch * 8) + 3 * align_up((size_t)spitch * 8) +
                   6 * align_up((size_t)n * 8) + 64 * 256;
    int rc = alloc_arena(ar, bytes);
    if (rc) return rc;
    const double *d_t, *d_y, *d_dy;
    if ((rc = stage_in(t, n, dev, ar, st, &d_t))) return rc;
    if ((rc = stage_in(y, n, dev, ar, st, &d_y))) return rc;
    if ((rc = stage_in(dy, n, dev, ar, st, &d_dy))) return rc;
    double* d_wr = ar.take<double>(n);
    double* d_w = ar.take<double>(n);
    double* d_wr2 = ar.take<double>(n);
    CurveInfo* d_info = ar.take<CurveInfo>(1);
    double* d_period = ar.take<double>(1);
    CU(cudaMemsetAsync(d_info, 0, sizeof(CurveInfo), st));
    CU(cudaMemcpyAsync(d_period, &period, sizeof(double), cudaMemcpyHostToDevice, st));
    launch_curve_pre(d_t, d_y, d_dy, (int)n, d_wr, d_w, d_wr2, d_info, st);
    CurveInfo info;
    CU(cudaMemcpyAsync(&info, d_info, sizeof(info), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    if (info.bad_curve) return GTLS_ENONFINITE;
    memset(&a, 0, sizeof(a));
    a.n = (int)n; a.tile = 1; a.p0 = 0; a.t = d_t; a.wr = d_wr; a.w = d_w; a.wr2 = d_wr2;
    a.periods = d_period; a.chi2_0 = &d_info->chi2_0; a.pitch = pitch; a.spitch = spitch;
    a.dt0 = o.dt0; a.uniform = 0;
    a.keys_a = ar.take<u64>(n); a.keys_b = ar.take<u64>(n); a.counts = ar.take<u32>(256ull * nt);
    a.perm = ar.take<u32>(n);
    SortScratch ssc;
    if (!take_sort_scratch(ar, 1, bucket_count_for((int)n), ssc)) return GTLS_ENOMEM;
    a.x1 = ar.take<double>(pitch); a.x0 = ar.take<double>(pitch);
    double* x2 = ar.take<double>(pitch);
    a.s1 = ar.take<double>(spitch); a.s0 = ar.take<double>(spitch);
    *d_s2 = ar.take<double>(spitch);
    if (!*d_s2) return GTLS_ENOMEM;
    run_fold_sort_scan(a, ssc, x2, *d_s2, (int)pad, false, nullptr, st, nullptr);
    return GTLS_OK;
}

int gtls_fold_scan(const double* t, const double* y, const double* dy, int64_t n, double period,
                   int64_t pad, const gtls_opts* opts, double* out_s1, double* out_s0,
                   double* out_s2) {
    g_cuda_err[0] = 0;
    const gtls_opts o = resolve_opts(opts);
    if (!t || !y || !dy || n < 1 || n > 0x3fffffff || pad < 0 || pad > n || !(period > 0.0)) return GTLS_EINVAL;
    CU(cudaSetDevice(o.device));
    cudaStream_t st = (cudaStream_t)o.stream;
    Arena ar;
    TileArgs a;
    double* d_s2 = nullptr;
    int rc = one_period_scan(t, y, dy, n, period, pad, o, ar, a, &d_s2);
    if (rc) return rc;
    const size_t cnt = (size_t)(n + pad + 1) * sizeof(double);
    const cudaMemcpyKind kind = o.pointers_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    if (out_s1) CU(cudaMemcpyAsync(out_s1, a.s1, cnt, kind, st));
    if (out_s0) CU(cudaMemcpyAsync(out_s0, a.s0, cnt, kind, st));
    if (out_s2) CU(cudaMemcpyAsync(out_s2, d_s2, cnt, kind, st));
    CU(cudaStreamSynchronize(st));
    CU(cudaGetLastError());
    return GTLS_OK;
}

int64_t gtls_window_chi2(const double* t, const double* y, const double* dy, int64_t n,
                         double period, double q, const double* tmpl, int32_t n_tmpl,
                         const gtls_opts* opts, int32_t* out_start, double* out_depth,
                         double* out_chi2_out, double* out_chi2_in) {
    g_cuda_err[0] = 0;
    const gtls_opts o = resolve_opts(opts);
    if (!t || !y || !dy || !tmpl || !out_start || !out_depth || !out_chi2_out || !out_chi2_in) return GTLS_EINVAL;
    if (n < 3 || n > 0x3fffffff || n_tmpl < 2 || !(period > 0.0) || !(q > 0.0) || !(q <= 0.5) || !(o.dt0 >= 0.0)) return GTLS_EINVAL;
    CU(cudaSetDevice(o.device));
    cudaStream_t st = (cudaStream_t)o.stream;
    const bool dev = o.pointers_on_device != 0;
    long long D = (long long)(q * (double)n);
    D = D < 1 ? 1 : (D > n - 1 ? n - 1 : D);
    long long stride = o.dt0 > 0.0 ? (long long)((double)D * o.dt0) : 1;
    if (stride < 1) stride = 1;
    const long long nW = (n + stride - 1) / stride;
    Arena ar;
    TileArgs a;
    double* d_s2 = nullptr;
    int rc = one_period_scan(t, y, dy, n, period, D, o, ar, a, &d_s2);
    if (rc) return rc;
    const double* d_tmpl;
    Arena ar2;
    if ((rc = alloc_arena(ar2, align_up(n_tmpl * 8) + 4 * align_up(nW * 8) + 16 * 256))) return rc;
    if ((rc = stage_in(tmpl, n_tmpl, dev, ar2, st, &d_tmpl))) return rc;
    a.tmpl = d_tmpl; a.n_tmpl = n_tmpl;
    int32_t* ds = dev ? out_start : ar2.take<int32_t>(nW);
    double* dd = dev ? out_depth : ar2.take<double>(nW);
    double* dco = dev ? out_chi2_out : ar2.take<double>(nW);
    double* dci = dev ? out_chi2_in : ar2.take<double>(nW);
    if (!dci) return GTLS_ENOMEM;
    launch_window_export(a, d_s2, q, ds, dd, dco, dci, st);
    if (!dev) {
        CU(cudaMemcpyAsync(out_start, ds, nW * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
        CU(cudaMemcpyAsync(out_depth, dd, nW * sizeof(double), cudaMemcpyDeviceToHost, st));
        CU(cudaMemcpyAsync(out_chi2_out, dco, nW * sizeof(double), cudaMemcpyDeviceToHost, st));
        CU(cudaMemcpyAsync(out_chi2_in, dci, nW * sizeof(double), cudaMemcpyDeviceToHost, st));
    }
    CU(cudaStreamSynchronize(st));
    CU(cudaGetLastError());
    return nW;
}

int gtls_sde(const double* chi2, int64_t n_per, const gtls_opts* opts, double* out_sde_raw,
             double* out_sde, gtls_summary* out_summary) {
    g_cuda_err[0] = 0;
    const gtls_opts o = resolve_opts(opts);
    if (!chi2 || n_per < 1) return GTLS_EINVAL;
    if (o.sde_kernel < 0 || (o.sde_kernel > 1 && o.sde_kernel % 2 == 0)) return GTLS_EINVAL;
    CU(cudaSetDevice(o.device));
    cudaStream_t st = (cudaStream_t)o.stream;
    const bool dev = o.pointers_on_device != 0;
    Arena ar;
    int rc = alloc_arena(ar, 3 * align_up(n_per * 8) + 8 * 256);
    if (rc) return rc;
    const double* d_chi2;
    if ((rc = stage_in(chi2, n_per, dev, ar, st, &d_chi2))) return rc;
    double* d_raw = (dev && out_sde_raw) ? out_sde_raw : ar.take<double>(n_per);
    double* d_sde = (dev && out_sde) ? out_sde : ar.take<double>(n_per);
    SdeScratch* d_sc = ar.take<SdeScratch>(1);
    if (!d_sc) return GTLS_ENOMEM;
    launch_sde(d_chi2, n_per, o.sde_kernel, d_raw, d_sde, d_sc, st, nullptr);
    SdeScratch sc;
    CU(cudaMemcpyAsync(&sc, d_sc, sizeof(sc), cudaMemcpyDeviceToHost, st));
    if (!dev) {
        if (out_sde_raw) CU(cudaMemcpyAsync(out_sde_raw, d_raw, n_per * 8, cudaMemcpyDeviceToHost, st));
        if (out_sde) CU(cudaMemcpyAsync(out_sde, d_sde, n_per * 8, cudaMemcpyDeviceToHost, st));
    }
    CU(cudaStreamSynchronize(st));
    CU(cudaGetLastError());
    if (out_summary) {
        memset(out_summary, 0, sizeof(*out_summary));
        out_summary->best_period_idx = sc.argmin;
        out_summary->chi2_min = sc.chi2_min;
        out_summary->sde_raw_max = sc.sde_raw_best;
        out_summary->sde_max = sc.sde_max;
        out_summary->sde_argmax = sc.sde_argmax;
    }
    return sc.degenerate ? GTLS_EDEGENERATE : GTLS_OK;
}

int gtls_search_two_stage(const double* t, const double* y, const double* dy, int64_t n,
                          const double* period_grid, int64_t n_per, const double* duration_grid,
                          int32_t n_dur, const double* tmpl, int32_t n_tmpl, const gtls_opts* opts,
                          int32_t n_refine, double* out_chi2, gtls_best* out_best, double* out_sde_raw,
                          double* out_sde, int64_t* out_refined, gtls_summary* out_summary) {
    g_cuda_err[0] = 0;
    const gtls_opts o = resolve_opts(opts);
    if (!t || !y || !dy || !period_grid || !duration_grid || !tmpl || !out_chi2 || !out_best) return GTLS_EINVAL;
    if (n < 3 || n_per < 1 || n_dur < 1 || n_tmpl < 2 || n_refine <= 0) return GTLS_EINVAL;
    CU(cudaSetDevice(o.device));
    cudaStream_t st = (cudaStream_t)o.stream;
    const bool dev = o.pointers_on_device != 0;
    const long long n_durs_total = o.dur_per_period ? n_per * (long long)n_dur : n_dur;
    const int K = (int)(n_refine < n_per ? n_refine : n_per);

    // device copies of everything (host mode), and the stage-2 scratch
    Arena ar;
    size_t bytes = align_up(n_per) + align_up((size_t)K * 8) * 3 + align_up((size_t)K * n_dur * 8) +
                   align_up((size_t)K * sizeof(gtls_best)) + 2 * align_up(n_per * 8) + 32 * 256;
    if (!dev)
        bytes += 3 * align_up(n * 8) + align_up(n_per * 8) + align_up(n_durs_total * 8) + align_up(n_tmpl * 8) +
                 align_up(n_per * 8) + align_up(n_per * sizeof(gtls_best));
    int rc = alloc_arena(ar, bytes);
    if (rc) return rc;
    const double *d_t, *d_y, *d_dy, *d_per, *d_dur, *d_tmpl;
    if ((rc = stage_in(t, n, dev, ar, st, &d_t))) return rc;
    if ((rc = stage_in(y, n, dev, ar, st, &d_y))) return rc;
    if ((rc = stage_in(dy, n, dev, ar, st, &d_dy))) return rc;
    if ((rc = stage_in(period_grid, n_per, dev, ar, st, &d_per))) return rc;
    if ((rc = stage_in(duration_grid, n_durs_total, dev, ar, st, &d_dur))) return rc;
    if ((rc = stage_in(tmpl, n_tmpl, dev, ar, st, &d_tmpl))) return rc;
    double* d_chi2 = dev ? out_chi2 : ar.take<double>(n_per);
    gtls_best* d_best = dev ? out_best : ar.take<gtls_best>(n_per);
    double* d_sde_raw = (dev && out_sde_raw) ? out_sde_raw : ar.take<double>(n_per);
    double* d_sde = (dev && out_sde) ? out_sde : ar.take<double>(n_per);
    unsigned char* d_mark = ar.take<unsigned char>(n_per);
    long long* d_sel = ar.take<long long>(K);
    double* d_per2 = ar.take<double>(K);
    double* d_dur2 = ar.take<double>((size_t)K * n_dur);
    double* d_chi2b = ar.take<double>(K);
    gtls_best* d_bestb = ar.take<gtls_best>(K);
    if (!d_bestb) return GTLS_ENOMEM;

    // ---- stage 1: coarse search over all periods ---------------------------------------------------
    gtls_opts o1 = o;
    o1.pointers_on_device = 1;
    o1.stats = nullptr;
    gtls_summary s1, s2, s3;
    memset(&s1, 0, sizeof(s1)); memset(&s2, 0, sizeof(s2)); memset(&s3, 0, sizeof(s3));
    rc = gtls_search(d_t, d_y, d_dy, n, d_per, n_per, d_dur, n_dur, d_tmpl, n_tmpl, &o1, d_chi2, d_best,
                     d_sde_raw, d_sde, &s1);
    int rc_final = rc;
    const bool refined = rc == GTLS_OK;
    if (refined) {
        // ---- stage 2: the K periods of highest SDE, every trial T0 -------------------------------------
        launch_topk_sde(d_sde, n_per, K, d_mark, d_sel, st);
        launch_gather_refine(d_per, d_dur, o.dur_per_period, n_dur, d_sel, K, d_per2, d_dur2, st);
        gtls_opts o2 = o1;
        o2.dt0 = 0.0;
        o2.dur_per_period = 1;
        o2.sde_kernel = 0;
        rc = gtls_search(d_t, d_y, d_dy, n, d_per2, K, d_dur2, n_dur, d_tmpl, n_tmpl, &o2, d_chi2b, d_bestb,
                         nullptr, nullptr, &s2);
        if (rc != GTLS_OK && rc != GTLS_EDEGENERATE) return rc;
        launch_merge_refined(d_sel, K, d_chi2b, d_bestb, d_chi2, d_best, st);
        rc_final = gtls_sde(d_chi2, n_per, &o1, d_sde_raw, d_sde, &s3);
        if (rc_final != GTLS_OK && rc_final != GTLS_EDEGENERATE) return rc_final;
    } else if (rc != GTLS_EDEGENERATE) {
        return rc;
    }
    if (out_summary) {
        *out_summary = s1;
        if (refined) {
            out_summary->best_period_idx = s3.best_period_idx;
            out_summary->chi2_min = s3.chi2_min;
            out_summary->sde_raw_max = s3.sde_raw_max;
            out_summary->sde_max = s3.sde_max;
            out_summary->sde_argmax = s3.sde_argmax;
            gtls_best b;
            double period = 0.0;
            CU(cudaMemcpyAsync(&b, d_best + s3.best_period_idx, sizeof(b), cudaMemcpyDeviceToHost, st));
            CU(cudaMemcpyAsync(&period, d_per + s3.best_period_idx, sizeof(double), cudaMemcpyDeviceToHost, st));
            CU(cudaStreamSynchronize(st));
            out_summary->best_dur_idx = b.dur_idx; out_summary->best_start = b.start;
            out_summary->best_period = period; out_summary->best_t0 = b.t0; out_summary->best_depth = b.depth;
        }
        out_summary->windows_evaluated = s1.windows_evaluated + s2.windows_evaluated;
    }
    const cudaMemcpyKind d2x = dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    if (out_refined && refined)
        CU(cudaMemcpyAsync(out_refined, d_sel, (size_t)K * sizeof(long long), d2x, st));
    if (!dev) {
        CU(cudaMemcpyAsync(out_chi2, d_chi2, n_per * sizeof(double), cudaMemcpyDeviceToHost, st));
        CU(cudaMemcpyAsync(out_best, d_best, n_per * sizeof(gtls_best), cudaMemcpyDeviceToHost, st));
        if (out_sde_raw) CU(cudaMemcpyAsync(out_sde_raw, d_sde_raw, n_per * sizeof(double), cudaMemcpyDeviceToHost, st));
        if (out_sde) CU(cudaMemcpyAsync(out_sde, d_sde, n_per * sizeof(double), cudaMemcpyDeviceToHost, st));
    }
    CU(cudaStreamSynchronize(st));
    CU(cudaGetLastError());
    return rc_final;
}

}  // extern "C"

// ---- trial grids on the device (paper section 2.2) --------------------------------------------------
namespace {
// SI constants: CODATA G, IAU nominal solar mass and radius.
constexpr double kGrav = 6.67430e-11, kMassSun = 1.98847e30, kRadiusSun = 6.957e8, kDaySeconds = 86400.0;
constexpr double kPi = 3.14159265358979323846;

// A/3, C and the real-valued N of Eq. 4-6.  Returns a gtls error code.
int ofir_constants(double span, double r_star, double m_star, double oversampling, double p_min,
                   double* a3, double* c, double* n_exact) {
    if (!(span > 0.0) || !(r_star > 0.0) || !(m_star > 0.0) || !(oversampling > 0.0) ||
        std::isinf(span) || std::isinf(r_star) || std::isinf(m_star) || std::isinf(oversampling) ||
        std::isnan(p_min) || std::isinf(p_min)) return GTLS_EINVAL;
    const double S = span * kDaySeconds;
    const double gm = kGrav * m_star * kMassSun;
    const double f_min = 2.0 / S;                                                          // Eq. 1
    double f_max;
    if (p_min > 0.0) f_max = 1.0 / (p_min * kDaySeconds);
    else { const double a_min = 3.0 * r_star * kRadiusSun; f_max = std::sqrt(gm / (a_min * a_min * a_min)) / (2.0 * kPi); }  // Eq. 3
    if (!(f_max > f_min)) return GTLS_EGRID;
    const double A = std::pow(2.0 * kPi, 2.0 / 3.0) / kPi * (r_star * kRadiusSun) / std::pow(gm, 1.0 / 3.0)
                     / (S * oversampling);                                                 // Eq. 5
    const double cf_min = std::pow(f_min, 1.0 / 3.0);
    *a3 = A / 3.0;
    *c = cf_min - A / 3.0;
    *n_exact = (std::pow(f_max, 1.0 / 3.0) - cf_min + A / 3.0) * 3.0 / A;                  // Eq. 6
    if (!(*n_exact >= 0.0) || *n_exact > 2147483647.0) return GTLS_EGRID;
    return GTLS_OK;
}

int batch_lanes(int n_curves) {
    static const int env = [] { const char* e = getenv("GTLS_BATCH_LANES"); return e ? atoi(e) : 0; }();
    int lanes = env > 0 ? env : 1;     // measured on c5: a c2-sized search fills the device; 2 lanes give 9.0-10.3 ms per
                                       // curve from run to run against a steady 9.1 ms for one lane, 4 / 8 lanes are 10 % slower
    if (lanes > 16) lanes = 16;
    return lanes < n_curves ? lanes : (n_curves < 1 ? 1 : n_curves);
}

// scratch of one lane: the largest gtls_workspace_bytes over the curves
size_t batch_lane_bytes(int32_t n_curves, const int64_t* co, const int64_t* po, int32_t n_dur, const gtls_opts* o) {
    size_t m = 0;
    for (int c = 0; c < n_curves; ++c) {
        const size_t b = gtls_workspace_bytes(co[c + 1] - co[c], po[c + 1] - po[c], n_dur, o);
        if (b > m) m = b;
    }
    return align_up(m);
}
}  // namespace

extern "C" {

int64_t gtls_period_grid_size(double span, double r_star, double m_star, double oversampling, double p_min) {
    double a3, c, n_exact;
    const int rc = ofir_constants(span, r_star, m_star, oversampling, p_min, &a3, &c, &n_exact);
    if (rc) return rc;
    const int64_t n = (int64_t)std::ceil(n_exact);
    return n < 1 ? GTLS_EGRID : n;
}

int gtls_period_grid(double span, double r_star, double m_star, double oversampling, double p_min,
                     const gtls_opts* opts, double* out_periods, int64_t n_per) {
    g_cuda_err[0] = 0;
    const gtls_opts o = resolve_opts(opts);
    double a3, c, n_exact;
    const int rc0 = ofir_constants(span, r_star, m_star, oversampling, p_min, &a3, &c, &n_exact);
    if (rc0) return rc0;
    if (!out_periods || n_per < 1 || n_per != (int64_t)std::ceil(n_exact)) return GTLS_EINVAL;
    CU(cudaSetDevice(o.device));
    cudaStream_t st = (cudaStream_t)o.stream;
    if (o.pointers_on_device) {
        launch_period_grid(a3, c, n_per, out_periods, st);
        CU(cudaGetLastError());
        return GTLS_OK;
    }
    Arena ar;
    int rc = alloc_arena(ar, align_up(n_per * 8) + 256);
    if (rc) return rc;
    double* d = ar.take<double>(n_per);
    launch_period_grid(a3, c, n_per, d, st);
    CU(cudaMemcpyAsync(out_periods, d, n_per * 8, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    CU(cudaGetLastError());
    return GTLS_OK;
}

int gtls_duration_grid(const double* periods, int64_t n_per, int32_t n_dur, double k_min, double k_max,
                       double q_cap, const gtls_opts* opts, double* out_durations) {
    g_cuda_err[0] = 0;
    const gtls_opts o = resolve_opts(opts);
    if (!periods || !out_durations || n_per < 1 || n_dur < 1 || n_dur > 4096) return GTLS_EINVAL;
    if (!(k_min > 0.0) || !(k_max >= k_min) || std::isinf(k_max) || !(q_cap > 0.0) || !(q_cap <= 0.5)) return GTLS_EINVAL;
    CU(cudaSetDevice(o.device));
    cudaStream_t st = (cudaStream_t)o.stream;
    const bool dev = o.pointers_on_device != 0;
    const size_t total = (size_t)n_per * n_dur;
    Arena ar;
    int rc = alloc_arena(ar, dev ? 512 : align_up(n_per * 8) + align_up(total * 8) + 1024);
    if (rc) return rc;
    const double* d_per;
    if ((rc = stage_in(periods, n_per, dev, ar, st, &d_per))) return rc;
    double* d_out = dev ? out_durations : ar.take<double>(total);
    int* d_bad = ar.take<int>(1);
    if (!d_bad) return GTLS_ENOMEM;
    CU(cudaMemsetAsync(d_bad, 0, sizeof(int), st));
    launch_duration_grid(d_per, n_per, n_dur, k_min, k_max, q_cap, d_out, d_bad, st);
    int bad = 0;
    CU(cudaMemcpyAsync(&bad, d_bad, sizeof(int), cudaMemcpyDeviceToHost, st));
    if (!dev) CU(cudaMemcpyAsync(out_durations, d_out, total * 8, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    CU(cudaGetLastError());
    return bad ? GTLS_EGRID : GTLS_OK;
}

size_t gtls_batch_workspace_bytes(int32_t n_curves, const int64_t* curve_offset,
                                  const int64_t* period_offset, int32_t n_dur, const gtls_opts* opts) {
    if (n_curves < 1 || !curve_offset || !period_offset) return 0;
    const gtls_opts o = resolve_opts(opts);
    const size_t lane = batch_lane_bytes(n_curves, curve_offset, period_offset, n_dur, &o);
    return lane ? (size_t)batch_lanes(n_curves) * lane + 256 : 0;
}

int gtls_search_batch(int32_t n_curves, const double* t, const double* y, const double* dy,
                      const int64_t* curve_offset, const double* period_grid,
                      const int64_t* period_offset, const double* duration_grid, int32_t n_dur,
                      const double* tmpl, int32_t n_tmpl, const gtls_opts* opts,
                      double* out_chi2, gtls_best* out_best, double* out_sde_raw, double* out_sde,
                      gtls_summary* out_summary, int32_t* out_status) {
    g_cuda_err[0] = 0;
    const gtls_opts o = resolve_opts(opts);
    if (n_curves < 1 || !t || !y || !dy || !curve_offset || !period_grid || !period_offset ||
        !duration_grid || !tmpl || !out_chi2 || n_dur < 1 || n_tmpl < 2) return GTLS_EINVAL;
    if (curve_offset[0] != 0 || period_offset[0] != 0) return GTLS_EINVAL;
    for (int c = 0; c < n_curves; ++c)
        if (curve_offset[c + 1] - curve_offset[c] < 3 || period_offset[c + 1] - period_offset[c] < 1) return GTLS_EINVAL;
    const int64_t n_total = curve_offset[n_curves], per_total = period_offset[n_curves];
    CU(cudaSetDevice(o.device));
    cudaStream_t st = (cudaStream_t)o.stream;
    const bool dev = o.pointers_on_device != 0;
    const int64_t durs_total = o.dur_per_period ? per_total * (int64_t)n_dur : n_dur;

    // host mode: everything is staged once; the curves then run on device pointers
    Arena io;
    if (!dev) {
        const size_t bytes = 3 * align_up(n_total * 8) + align_up(per_total * 8) + align_up(durs_total * 8) +
                             align_up(n_tmpl * 8) + 3 * align_up(per_total * 8) +
                             align_up(per_total * sizeof(gtls_best)) + 16 * 256;
        int rc = alloc_arena(io, bytes);
        if (rc) return rc;
    }
    const double *d_t, *d_y, *d_dy, *d_per, *d_dur, *d_tmpl;
    int rc;
    if ((rc = stage_in(t, n_total, dev, io, st, &d_t))) return rc;
    if ((rc = stage_in(y, n_total, dev, io, st, &d_y))) return rc;
    if ((rc = stage_in(dy, n_total, dev, io, st, &d_dy))) return rc;
    if ((rc = stage_in(period_grid, per_total, dev, io, st, &d_per))) return rc;
    if ((rc = stage_in(duration_grid, durs_total, dev, io, st, &d_dur))) return rc;
    if ((rc = stage_in(tmpl, n_tmpl, dev, io, st, &d_tmpl))) return rc;
    double* d_chi2 = dev ? out_chi2 : io.take<double>(per_total);
    gtls_best* d_best = dev ? out_best : (out_best ? io.take<gtls_best>(per_total) : nullptr);
    double* d_raw = dev ? out_sde_raw : (out_sde_raw ? io.take<double>(per_total) : nullptr);
    double* d_sde = dev ? out_sde : (out_sde ? io.take<double>(per_total) : nullptr);
    if (!d_chi2 || (out_best && !d_best) || (out_sde_raw && !d_raw) || (out_sde && !d_sde)) return GTLS_ENOMEM;

    // scratch: one slice per lane
    const int lanes = batch_lanes(n_curves);
    gtls_opts sized = o;                      // the per-curve tile choice without the caller's scratch
    sized.workspace = nullptr; sized.workspace_bytes = 0;
    size_t lane_bytes = batch_lane_bytes(n_curves, curve_offset, period_offset, n_dur, &sized);
    if (!lane_bytes) return GTLS_EINVAL;
    Arena ws;
    if (o.workspace) {
        if (((uintptr_t)o.workspace & 255) != 0) return GTLS_EINVAL;
        if (o.workspace_bytes < (size_t)lanes * lane_bytes) return GTLS_ENOMEM;
        ws.base = (char*)o.workspace; ws.size = o.workspace_bytes; ws.owned = false;
    } else {
        size_t free_b = 0, total_b = 0;
        if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess && (size_t)lanes * lane_bytes > free_b / 2)
            lane_bytes = (free_b / 2 / lanes) & ~(size_t)255;      // gtls_search shrinks its tile to fit
        if ((rc = alloc_arena(ws, (size_t)lanes * lane_bytes + 256))) return rc;
    }

    cudaEvent_t ev_in = nullptr;
    CU(cudaEventCreateWithFlags(&ev_in, cudaEventDisableTiming));
    CU(cudaEventRecord(ev_in, st));
    std::vector<int> status((size_t)n_curves, GTLS_OK);
    std::vector<cudaEvent_t> ev_done((size_t)lanes, nullptr);
    std::vector<int> lane_rc((size_t)lanes, GTLS_OK);
    std::vector<std::thread> workers;
    auto lane_body = [&](int lane) {
            cudaStream_t ls = nullptr;
            if (cudaSetDevice(o.device) != cudaSuccess ||
                cudaStreamCreateWithFlags(&ls, cudaStreamNonBlocking) != cudaSuccess ||
                cudaEventCreateWithFlags(&ev_done[lane], cudaEventDisableTiming) != cudaSuccess ||
                cudaStreamWaitEvent(ls, ev_in, 0) != cudaSuccess) {
                lane_rc[lane] = GTLS_ECUDA;
                for (int c = lane; c < n_curves; c += lanes) status[c] = GTLS_ECUDA;
                if (ls) cudaStreamDestroy(ls);
                return;
            }
            gtls_opts lo = o;
            lo.pointers_on_device = 1;
            lo.stream = (void*)ls;
            lo.workspace = ws.base + (size_t)lane * lane_bytes;
            lo.workspace_bytes = lane_bytes;
            lo.stats = nullptr;
            for (int c = lane; c < n_curves; c += lanes) {
                const int64_t c0 = curve_offset[c], p0 = period_offset[c];
                status[c] = gtls_search(d_t + c0, d_y + c0, d_dy + c0, curve_offset[c + 1] - c0,
                                        d_per + p0, period_offset[c + 1] - p0,
                                        o.dur_per_period ? d_dur + p0 * n_dur : d_dur, n_dur, d_tmpl, n_tmpl, &lo,
                                        d_chi2 + p0, d_best ? d_best + p0 : nullptr, d_raw ? d_raw + p0 : nullptr,
                                        d_sde ? d_sde + p0 : nullptr, out_summary ? out_summary + c : nullptr);
            }
            cudaEventRecord(ev_done[lane], ls);
            cudaStreamSynchronize(ls);
            cudaStreamDestroy(ls);
    };
    for (int lane = 1; lane < lanes; ++lane) {
        try { workers.emplace_back(lane_body, lane); }
        catch (...) { lane_body(lane); }          // no thread to be had: the lane runs here, in turn
    }
    lane_body(0);                                 // the calling thread is lane 0
    for (auto& w : workers) w.join();
    for (int lane = 0; lane < lanes; ++lane)
        if (ev_done[lane]) { cudaStreamWaitEvent(st, ev_done[lane], 0); cudaEventDestroy(ev_done[lane]); }
    cudaEventDestroy(ev_in);
    int first = GTLS_OK;
    for (int c = 0; c < n_curves; ++c) {
        if (out_status) out_status[c] = status[c];
        if (first == GTLS_OK && status[c] != GTLS_OK && status[c] != GTLS_EDEGENERATE) first = status[c];
    }
    if (!dev) {
        CU(cudaMemcpyAsync(out_chi2, d_chi2, per_total * sizeof(double), cudaMemcpyDeviceToHost, st));
        if (out_best) CU(cudaMemcpyAsync(out_best, d_best, per_total * sizeof(gtls_best), cudaMemcpyDeviceToHost, st));
        if (out_sde_raw) CU(cudaMemcpyAsync(out_sde_raw, d_raw, per_total * sizeof(double), cudaMemcpyDeviceToHost, st));
        if (out_sde) CU(cudaMemcpyAsync(out_sde, d_sde, per_total * sizeof(double), cudaMemcpyDeviceToHost, st));
    }
    CU(cudaStreamSynchronize(st));
    return first;
}

}  // extern "C"
