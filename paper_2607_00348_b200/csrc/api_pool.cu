// Device block pool, arena allocation, option defaults, the per-thread side streams and the small
// informational entry points of the C ABI (include/gtls.h).
#include "api_common.cuh"

namespace gtls {
namespace api {

char* cuda_err_buf() {
    thread_local char buf[512] = "";
    return buf;
}
int cuda_fail(cudaError_t e, const char* what) {
    snprintf(cuda_err_buf(), 512, "%s: %s (%s)", what, cudaGetErrorString(e), cudaGetErrorName(e));
    return GTLS_ECUDA;
}

namespace {
// Device blocks the library allocated itself are kept in a small pool between calls (cudaMalloc and
// cudaFree of a few GB cost milliseconds each and cudaFree synchronises the device: half of the end-to-end
// time of a short light curve through host buffers).  At most kPoolSlots free blocks, each at most
// GTLS_CACHE_MB (default 8192) MiB; gtls_release_cache() frees them; GTLS_CACHE_MB=0 switches the pool off.
constexpr int kPoolSlots = 4;
struct PoolBlock { char* base; size_t size; int dev; };
std::mutex g_pool_mu;
PoolBlock g_pool[kPoolSlots] = {};
}  // namespace
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

void pool_release_all() {
    std::lock_guard<std::mutex> lk(g_pool_mu);
    for (auto& b : g_pool) { if (b.base) cudaFree(b.base); b = PoolBlock{}; }
}

int alloc_arena(Arena& ar, size_t bytes) {
    size_t got = 0;
    if (char* p = pool_take(bytes, &got)) { ar.base = p; ar.size = got; ar.off = 0; ar.owned = true; return GTLS_OK; }
    if (pool_cap() && bytes <= pool_cap()) bytes = align_up(bytes + bytes / 16, 2u << 20);   // slack: the next, slightly larger request fits too
    cudaError_t e = cudaMalloc((void**)&ar.base, bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        pool_release_all();                  // the pool may hold what this request needs
        e = cudaMalloc((void**)&ar.base, bytes);
    }
    if (e != cudaSuccess) { cudaGetLastError(); ar.base = nullptr; snprintf(cuda_err_buf(), 512, "cudaMalloc(%zu): %s", bytes, cudaGetErrorString(e)); return GTLS_ENOMEM; }
    ar.size = bytes; ar.off = 0; ar.owned = true;
    return GTLS_OK;
}

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

}  // namespace api

SideStream* side_stream(int which) {
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

}  // namespace gtls

using namespace gtls;

extern "C" {

void gtls_opts_default(gtls_opts* o) {
    if (!o) return;
    memset(o, 0, sizeof(*o));
    o->struct_size = sizeof(gtls_opts);
    o->dt0 = 0.05;
    o->sde_kernel = 151;
}

const char* gtls_version(void) { return "gtls-b200 0.1.0 (sm_100a)"; }

void gtls_release_cache(void) { api::pool_release_all(); }
const char* gtls_last_cuda_error(void) { return api::cuda_err_buf(); }

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

}  // extern "C"
