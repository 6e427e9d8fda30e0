// gtls_search_static: the fused small-N search (small.cu) for callers that cannot
// allocate -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// Every byte of scratch the search needs lives in ONE file-scope device array of a fixed, modest size
// (kStaticBytes, ~263 KB; every GPU that loads the library holds it until exit).  The entry point calls no
// cudaMalloc, cudaFree or allocating library routine and never touches the library's block pool; inputs and
// outputs are the caller's device arrays.  All calls (from any thread, on any stream) share the array, which
// keeps the previous call's contents: what must start at zero is cleared on the call's stream, and two calls
// that overlap on the same GPU race -- the caller serialises them.
//
// In host code the array's NAME is a host-side stand-in, not a device address; the address is taken once per
// device with cudaGetSymbolAddress (with that device current) and only that pointer is handed to kernels.
#include <mutex>

#include "api_common.cuh"

using namespace gtls;
using namespace gtls::api;

namespace {

constexpr int kStaticMaxN = GTLS_STATIC_MAX_N;            // light-curve points
constexpr int kStaticMaxD = kStaticMaxN / 2;              // window length: q <= 0.5
constexpr size_t kOffWr = 0;                                                   // double[kStaticMaxN]  w r
constexpr size_t kOffW = kOffWr + (size_t)kStaticMaxN * 8;                    // double[kStaticMaxN]  w
constexpr size_t kOffWr2 = kOffW + (size_t)kStaticMaxN * 8;                   // double[kStaticMaxN]  w r^2
constexpr size_t kOffGtab = kOffWr2 + (size_t)kStaticMaxN * 8;                // double[2 (kStaticMaxD + 1)] template sums
constexpr size_t kOffInfo = (kOffGtab + 2 * (size_t)(kStaticMaxD + 1) * 8 + 255) / 256 * 256;   // CurveInfo
constexpr size_t kOffSde = kOffInfo + 256;                                     // SdeScratch
constexpr size_t kOffCnt = kOffSde + 256;                                      // u64[2] window counters + u64 work queue
constexpr size_t kOffOffs = kOffCnt + 256;                                     // long long[4] curve / period offsets
constexpr size_t kStaticBytes = kOffOffs + 256;
static_assert(sizeof(CurveInfo) <= 256 && sizeof(SdeScratch) <= 256, "scratch slots");

static __device__ __align__(256) unsigned char g_static_scratch[kStaticBytes];

// Device address of the scratch array on `device` (which must be current): looked up once per device.
int static_scratch_ptr(int device, unsigned char** out) {
    constexpr int kMaxDevices = 64;
    static std::mutex mu;
    static unsigned char* ptr[kMaxDevices] = {};
    if (device < 0 || device >= kMaxDevices) return GTLS_EINVAL;
    std::lock_guard<std::mutex> lk(mu);
    if (!ptr[device]) {
        unsigned char* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
        if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(g_static_scratch)");
        if (!p) return GTLS_ECUDA;
        ptr[device] = p;
    }
    *out = ptr[device];
    return GTLS_OK;
}

// refusals carry their reason in the text gtls_last_cuda_error() returns
int refuse(int code, const char* fmt, long long a, long long b) {
    snprintf(cuda_err_buf(), 512, fmt, a, b);
    return code;
}
int refuse(int code, const char* msg) {
    snprintf(cuda_err_buf(), 512, "%s", msg);
    return code;
}

}  // namespace

extern "C" {

size_t gtls_static_scratch_bytes(void) { return kStaticBytes; }

int gtls_search_static(const double* t, const double* y, const double* dy, int64_t n,
                       const double* period_grid, int64_t n_per, const double* duration_grid,
                       int32_t n_dur, const double* tmpl, int32_t n_tmpl, const gtls_opts* opts,
                       double* out_chi2, gtls_best* out_best, double* out_sde_raw, double* out_sde,
                       gtls_summary* out_summary) {
    cuda_err_buf()[0] = 0;
    const gtls_opts o = resolve_opts(opts);
    if (!t || !y || !dy || !period_grid || !duration_grid || !tmpl) return GTLS_EINVAL;
    if (!out_chi2 || !out_best || !out_sde_raw || !out_sde) return GTLS_EINVAL;      // no scratch to stand in for them
    if (n < 3 || n_per < 1 || n_dur < 1 || n_tmpl < 2) return GTLS_EINVAL;
    if (!(o.dt0 >= 0.0) || o.sde_kernel < 0 || (o.sde_kernel > 1 && o.sde_kernel % 2 == 0)) return GTLS_EINVAL;
    if (n > kStaticMaxN)
        return refuse(GTLS_EUNSUPPORTED, "gtls_search_static: n = %lld exceeds the static scratch maximum of %lld points",
                      (long long)n, (long long)kStaticMaxN);
    if (n_dur > 32)
        return refuse(GTLS_EUNSUPPORTED, "gtls_search_static: n_dur = %lld exceeds the fused kernel's maximum of %lld",
                      (long long)n_dur, 32);
    if (o.top_k != 0 || o.chi2_fp32 != 0)
        return refuse(GTLS_EUNSUPPORTED, "gtls_search_static: top_k (%lld) / chi2_fp32 (%lld) are not offered by the fused kernel",
                      (long long)o.top_k, (long long)o.chi2_fp32);
    CU(cudaSetDevice(o.device));
    cudaStream_t st = (cudaStream_t)o.stream;
    unsigned char* base = nullptr;
    int rc = static_scratch_ptr(o.device, &base);
    if (rc) return rc;
    double* d_wr = reinterpret_cast<double*>(base + kOffWr);
    double* d_w = reinterpret_cast<double*>(base + kOffW);
    double* d_wr2 = reinterpret_cast<double*>(base + kOffWr2);
    double* d_gtab = reinterpret_cast<double*>(base + kOffGtab);
    CurveInfo* d_info = reinterpret_cast<CurveInfo*>(base + kOffInfo);
    SdeScratch* d_sc = reinterpret_cast<SdeScratch*>(base + kOffSde);
    unsigned long long* d_cnt = reinterpret_cast<unsigned long long*>(base + kOffCnt);
    long long* d_off = reinterpret_cast<long long*>(base + kOffOffs);
    const long long n_durs_total = o.dur_per_period ? n_per * (long long)n_dur : n_dur;

    // the array keeps the last call's contents: flags, counters and the work queue start at zero
    CU(cudaMemsetAsync(d_info, 0, sizeof(CurveInfo), st));
    CU(cudaMemsetAsync(d_cnt, 0, 3 * sizeof(unsigned long long), st));
    // a0 + validation (one host synchronisation, as in gtls_search)
    launch_curve_pre(t, y, dy, (int)n, d_wr, d_w, d_wr2, d_info, st);
    launch_grid_check(period_grid, n_per, duration_grid, n_durs_total, d_info, st);
    CurveInfo info;
    CU(cudaMemcpyAsync(&info, d_info, sizeof(info), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    CU(cudaGetLastError());
    if (info.bad_curve) return GTLS_ENONFINITE;
    if (info.bad_period || info.bad_duration) return GTLS_EGRID;
    if (info.w_min != info.w_max)
        return refuse(GTLS_EUNSUPPORTED, "gtls_search_static: dy is not uniform (the fused kernel needs one common weight)");
    long long dmax = (long long)(info.q_max * (double)n);
    dmax = dmax < 1 ? 1 : (dmax > n - 1 ? n - 1 : dmax);
    if (dmax > kStaticMaxD || !small_path_fits((int)n, (int)dmax, n_dur, o.dt0))
        return refuse(GTLS_EUNSUPPORTED, "gtls_search_static: n = %lld with windows of up to %lld points does not fit the fused kernel "
                      "(shared memory of one CTA, or a window class stride above 31 columns at this dt0)", (long long)n, dmax);
    launch_gtab(tmpl, n_tmpl, (int)dmax, d_gtab, st);
    const long long h_off[4] = {0, (long long)n, 0, (long long)n_per};
    CU(cudaMemcpyAsync(d_off, h_off, sizeof(h_off), cudaMemcpyHostToDevice, st));
    SmallArgs sa;
    memset(&sa, 0, sizeof(sa));
    sa.n_items = n_per; sa.n_dur = n_dur; sa.n_tmpl = n_tmpl; sa.dur_per_period = o.dur_per_period; sa.dt0 = o.dt0;
    sa.curve_off = d_off; sa.per_off = d_off + 2;
    sa.t = t; sa.wr = d_wr; sa.info = d_info; sa.periods = period_grid; sa.durs = duration_grid; sa.tmpl = tmpl;
    sa.gtab = d_gtab; sa.out_chi2 = out_chi2; sa.out_best = out_best; sa.counters = d_cnt; sa.queue = d_cnt + 2;
    int sms = 0;
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, o.device));
    const int ce = launch_tls_small(sa, (int)n, (int)dmax, sms, st);
    if (ce != 0) return cuda_fail((cudaError_t)ce, "k_tls_small");
    // a9
    launch_sde(out_chi2, n_per, o.sde_kernel, out_sde_raw, out_sde, d_sc, st, nullptr);
    SdeScratch sc;
    unsigned long long counters[2];
    CU(cudaMemcpyAsync(&sc, d_sc, sizeof(sc), cudaMemcpyDeviceToHost, st));
    CU(cudaMemcpyAsync(counters, d_cnt, sizeof(counters), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));               // (also keeps h_off alive until its copy has been taken)
    CU(cudaGetLastError());
    if (out_summary) {
        gtls_best b;
        double period = 0.0;
        CU(cudaMemcpyAsync(&b, out_best + sc.argmin, sizeof(b), cudaMemcpyDeviceToHost, st));
        CU(cudaMemcpyAsync(&period, period_grid + sc.argmin, sizeof(double), cudaMemcpyDeviceToHost, st));
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
    return sc.degenerate ? GTLS_EDEGENERATE : GTLS_OK;
}

}  // extern "C"
