// Trial grids built on the device (paper section 2.2): Ofir period grid (Eq. 1-6) and the per-period
// duration grid (Eq. 8-9, reading G12).
#include "api_common.cuh"

using namespace gtls;
using namespace gtls::api;

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
    api::cuda_err_buf()[0] = 0;
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
    api::cuda_err_buf()[0] = 0;
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

}  // extern "C"
