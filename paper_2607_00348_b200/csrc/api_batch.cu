// Survey mode (BASELINE.json config 5): gtls_search_batch over concatenated light curves.
#include <algorithm>
#include <thread>
#include <vector>

#include "api_common.cuh"

using namespace gtls;
using namespace gtls::api;

namespace {
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

// Fused small-N path over the whole batch (small.cu): ONE kernel whose work items are the (curve, period)
// pairs of every curve, no per-curve host synchronisation.  Applies when every curve passes validation, has
// uniform dy and fits the fused kernel's limits; returns false (nothing written) when it does not, and the
// caller runs the curves one by one through gtls_search.
bool fused_batch(const gtls_opts& o, int32_t n_curves, const int64_t* curve_offset, const int64_t* period_offset,
                 const double* d_t, const double* d_y, const double* d_dy, const double* d_per, const double* d_dur,
                 int32_t n_dur, const double* d_tmpl, int32_t n_tmpl, double* d_chi2, gtls_best* d_best_out,
                 double* d_raw_out, double* d_sde_out, gtls_summary* out_summary, int32_t* out_status,
                 cudaStream_t st, int* rc_out) {
    if (o.path == 2 || o.top_k != 0 || o.chi2_fp32 != 0 || n_dur > 32) return false;
    const int64_t n_total = curve_offset[n_curves], per_total = period_offset[n_curves];
    int64_t n_max = 0;
    for (int c = 0; c < n_curves; ++c) n_max = std::max<int64_t>(n_max, curve_offset[c + 1] - curve_offset[c]);
    if (n_max > 65535) return false;
    Arena ar;
    const size_t bytes = 3 * align_up(n_total * 8) + align_up(n_curves * sizeof(CurveInfo)) +
                         align_up(n_curves * sizeof(SdeScratch)) + align_up(2 * n_curves * sizeof(unsigned long long)) +
                         2 * align_up((n_curves + 1) * sizeof(long long)) + align_up(n_curves * sizeof(gtls_summary)) +
                         align_up(2 * (size_t)(n_max + 2) * 8) + 2 * align_up(per_total * 8) +
                         align_up(per_total * sizeof(gtls_best)) + 32 * 256;
    if (alloc_arena(ar, bytes) != GTLS_OK) return false;
    double* d_wr = ar.take<double>(n_total);
    double* d_w = ar.take<double>(n_total);
    double* d_wr2 = ar.take<double>(n_total);
    CurveInfo* d_info = ar.take<CurveInfo>(n_curves);
    SdeScratch* d_sc = ar.take<SdeScratch>(n_curves);
    unsigned long long* d_cnt = ar.take<unsigned long long>(2 * (size_t)n_curves + 1);   // counters + the work queue
    long long* d_coff = ar.take<long long>(n_curves + 1);
    long long* d_poff = ar.take<long long>(n_curves + 1);
    gtls_summary* d_summ = ar.take<gtls_summary>(n_curves);
    double* d_raw = d_raw_out ? d_raw_out : ar.take<double>(per_total);
    double* d_sde = d_sde_out ? d_sde_out : ar.take<double>(per_total);
    gtls_best* d_best = d_best_out ? d_best_out : ar.take<gtls_best>(per_total);
    if (!d_best) return false;
    auto fail = [&](int rc) { *rc_out = rc; return true; };
    static_assert(sizeof(long long) == sizeof(int64_t), "offset arrays are copied as they are");
    if (cudaMemcpyAsync(d_coff, curve_offset, (n_curves + 1) * sizeof(long long), cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(d_poff, period_offset, (n_curves + 1) * sizeof(long long), cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaMemsetAsync(d_info, 0, n_curves * sizeof(CurveInfo), st) != cudaSuccess ||
        cudaMemsetAsync(d_cnt, 0, (2 * (size_t)n_curves + 1) * sizeof(unsigned long long), st) != cudaSuccess)
        return fail(cuda_fail(cudaGetLastError(), "fused batch set-up"));
    launch_batch_pre(n_curves, d_t, d_y, d_dy, d_coff, d_per, d_poff, d_dur, n_dur, o.dur_per_period, d_wr, d_w, d_wr2,
                     d_info, st);
    std::vector<CurveInfo> info((size_t)n_curves);
    if (cudaMemcpyAsync(info.data(), d_info, n_curves * sizeof(CurveInfo), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess)
        return fail(cuda_fail(cudaGetLastError(), "fused batch validation"));
    // the ONE host synchronisation of the batch: validation flags, uniform dy, the largest duration
    int d_max = 1;
    for (int c = 0; c < n_curves; ++c) {
        const int64_t n = curve_offset[c + 1] - curve_offset[c];
        if (info[c].bad_curve || info[c].bad_period || info[c].bad_duration || info[c].w_min != info[c].w_max) {
            ar.idle = true;
            return false;                      // a curve needs the general path or fails validation: one by one
        }
        long long dm = (long long)(info[c].q_max * (double)n);
        dm = dm < 1 ? 1 : (dm > n - 1 ? n - 1 : dm);
        d_max = std::max(d_max, (int)dm);
    }
    if (!small_path_fits((int)n_max, d_max, n_dur, o.dt0)) {
        ar.idle = true;
        if (o.path == 1) return fail(GTLS_EUNSUPPORTED);
        return false;
    }
    double* d_gtab = ar.take<double>(2 * (size_t)(d_max + 1));
    if (!d_gtab) { ar.idle = true; return false; }
    launch_gtab(d_tmpl, n_tmpl, d_max, d_gtab, st);
    SmallArgs sa;
    memset(&sa, 0, sizeof(sa));
    sa.n_items = per_total; sa.n_dur = n_dur; sa.n_tmpl = n_tmpl; sa.dur_per_period = o.dur_per_period; sa.dt0 = o.dt0;
    sa.curve_off = d_coff; sa.per_off = d_poff; sa.t = d_t; sa.wr = d_wr; sa.info = d_info;
    sa.periods = d_per; sa.durs = d_dur; sa.tmpl = d_tmpl; sa.gtab = d_gtab;
    sa.out_chi2 = d_chi2; sa.out_best = d_best; sa.counters = d_cnt; sa.queue = d_cnt + 2 * (size_t)n_curves;
    int sms = 0;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, o.device);
    const int ce = launch_tls_small(sa, (int)n_max, d_max, sms, st);
    if (ce != 0) return fail(cuda_fail((cudaError_t)ce, "k_tls_small"));
    // a9 per curve (the moving median needs a curve's own neighbours), then every summary in one kernel
    for (int c = 0; c < n_curves; ++c) {
        const int64_t p0 = period_offset[c];
        launch_sde(d_chi2 + p0, period_offset[c + 1] - p0, o.sde_kernel, d_raw + p0, d_sde + p0, d_sc + c, st, nullptr);
    }
    launch_batch_summary(n_curves, d_poff, d_sc, d_best, d_per, d_info, d_cnt, d_summ, st);
    std::vector<SdeScratch> sc((size_t)n_curves);
    if (cudaMemcpyAsync(sc.data(), d_sc, n_curves * sizeof(SdeScratch), cudaMemcpyDeviceToHost, st) != cudaSuccess)
        return fail(cuda_fail(cudaGetLastError(), "fused batch epilogue"));
    if (out_summary &&
        cudaMemcpyAsync(out_summary, d_summ, n_curves * sizeof(gtls_summary), cudaMemcpyDeviceToHost, st) != cudaSuccess)
        return fail(cuda_fail(cudaGetLastError(), "fused batch summaries"));
    if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess)
        return fail(cuda_fail(cudaGetLastError(), "fused batch"));
    ar.idle = true;
    for (int c = 0; c < n_curves; ++c)
        if (out_status) out_status[c] = sc[c].degenerate ? GTLS_EDEGENERATE : GTLS_OK;
    *rc_out = GTLS_OK;
    return true;
}
}  // namespace

extern "C" {

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
    api::cuda_err_buf()[0] = 0;
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

    // a caller-owned scratch is checked against gtls_batch_workspace_bytes whichever path runs
    const int lanes = batch_lanes(n_curves);
    gtls_opts sized = o;                      // the per-curve tile choice without the caller's scratch
    sized.workspace = nullptr; sized.workspace_bytes = 0;
    size_t lane_bytes = batch_lane_bytes(n_curves, curve_offset, period_offset, n_dur, &sized);
    if (!lane_bytes) return GTLS_EINVAL;
    if (o.workspace) {
        if (((uintptr_t)o.workspace & 255) != 0) return GTLS_EINVAL;
        if (o.workspace_bytes < (size_t)lanes * lane_bytes) return GTLS_ENOMEM;
    }
    // ---- fused small-N path: one kernel over every (curve, period) of the batch -------------------
    if (o.sde_kernel < 0 || (o.sde_kernel > 1 && o.sde_kernel % 2 == 0) || !(o.dt0 >= 0.0)) return GTLS_EINVAL;
    {
        int frc = GTLS_OK;
        if (fused_batch(o, n_curves, curve_offset, period_offset, d_t, d_y, d_dy, d_per, d_dur, n_dur, d_tmpl, n_tmpl,
                        d_chi2, d_best, d_raw, d_sde, out_summary, out_status, st, &frc)) {
            if (frc != GTLS_OK) return frc;
            if (!dev) {
                CU(cudaMemcpyAsync(out_chi2, d_chi2, per_total * sizeof(double), cudaMemcpyDeviceToHost, st));
                if (out_best) CU(cudaMemcpyAsync(out_best, d_best, per_total * sizeof(gtls_best), cudaMemcpyDeviceToHost, st));
                if (out_sde_raw) CU(cudaMemcpyAsync(out_sde_raw, d_raw, per_total * sizeof(double), cudaMemcpyDeviceToHost, st));
                if (out_sde) CU(cudaMemcpyAsync(out_sde, d_sde, per_total * sizeof(double), cudaMemcpyDeviceToHost, st));
                CU(cudaStreamSynchronize(st));
            }
            io.idle = true;
            return GTLS_OK;
        }
        if (o.path == 1) return GTLS_EUNSUPPORTED;
    }

    // scratch: one slice per lane
    Arena ws;
    if (o.workspace) {
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
