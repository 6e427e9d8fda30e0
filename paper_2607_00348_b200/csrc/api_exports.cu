// Debug / parity exports of the C ABI: gtls_fold_sort (a1-a2), gtls_fold_scan (a3-a4), gtls_window_chi2
// (a5-a7 per window) and gtls_sde (a9 alone).
#include "api_common.cuh"

using namespace gtls;
using namespace gtls::api;

extern "C" {

int gtls_fold_sort(const double* t, int64_t n, const double* periods, int64_t n_per,
                   const gtls_opts* opts, double* out_phase, int32_t* out_perm) {
    api::cuda_err_buf()[0] = 0;
    const gtls_opts o = resolve_opts(opts);
    if (!t || !periods || !out_perm || n < 1 || n > 0x3fffffff || n_per < 1) return GTLS_EINVAL;
    CU(cudaSetDevice(o.device));
    cudaStream_t st = (cudaStream_t)o.stream;
    const bool dev = o.pointers_on_device != 0;
    const int nt = (int)((n + kRadixTile - 1) / kRadixTile);
    const size_t per_period = 2 * n * sizeof(u64) + 256ull * nt * sizeof(u32) + n * sizeof(u32) +
                              sort_scratch_bytes(n) + 1024 +
                              (dev ? 0 : n * (sizeof(double) + sizeof(int32_t))) + 1024;
    long long tile = (long long)((1ull << 30) / per_period);
    if (tile > 8192) tile = 8192;                               // (a tile is gridDim.y of the sort kernels: <= 65535)
    if (o.period_tile > 0) tile = o.period_tile < 65535 ? o.period_tile : 65535;
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
    if (!take_sort_scratch(ar, (size_t)tile, (int)n, ssc)) return GTLS_ENOMEM;
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
    if (!take_sort_scratch(ar, 1, (int)n, ssc)) return GTLS_ENOMEM;
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
    api::cuda_err_buf()[0] = 0;
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
    api::cuda_err_buf()[0] = 0;
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
    api::cuda_err_buf()[0] = 0;
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

}  // extern "C"
