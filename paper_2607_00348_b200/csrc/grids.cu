// Trial grids built on the device: the Ofir cubic frequency sampling
// of the period grid (Eq. 4) and the per-period log-spaced duration fractions between the
// empirical envelopes of Eq. 8-9 with the cap of PAPER.md:159 (reading G12).
// The scalar constants A and C of Eq. 5 are computed once per call on the host (gtls_api.cu).
#include "gtls_internal.cuh"

namespace gtls {
namespace {

constexpr double kSecondsPerDay = 86400.0;

// f_i = (A/3 i + C)^3, i = 1..N; out[i-1] = 1 / f_i in days.  Explicit round-to-nearest operations:
// no FMA contraction, so the values do not depend on how the compiler fuses the cube.
__global__ void __launch_bounds__(256) k_period_grid(double a3, double c, long long n_per, double* __restrict__ out) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= n_per) return;
    const double x = __dadd_rn(__dmul_rn(a3, (double)(i + 1)), c);
    const double f = __dmul_rn(__dmul_rn(x, x), x);
    out[i] = __ddiv_rn(__ddiv_rn(1.0, f), kSecondsPerDay);
}

// One thread per (period, duration index): q = exp((1-x) ln q_lo + x ln q_hi), x = j/(n_dur-1),
// q_lo = min(k_min P^(-2/3), cap), q_hi = min(k_max P^(-2/3), cap), P in seconds.
// A period that is not finite or <= 0 raises *bad (the row is filled with NaN).
__global__ void __launch_bounds__(256) k_duration_grid(const double* __restrict__ periods, long long n_per, int n_dur,
                                                       double k_min, double k_max, double q_cap,
                                                       double* __restrict__ out, int* __restrict__ bad) {
    const long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (idx >= n_per * n_dur) return;
    const long long ip = idx / n_dur;
    const int j = (int)(idx - ip * n_dur);
    const double p = periods[ip];
    if (!(p > 0.0) || isinf(p)) {
        if (j == 0) atomicAdd(bad, 1);
        out[idx] = __longlong_as_double(0x7ff8000000000000LL);
        return;
    }
    const double scale = pow(p * kSecondsPerDay, -2.0 / 3.0);
    const double q_lo = fmin(k_min * scale, q_cap), q_hi = fmin(k_max * scale, q_cap);
    const double x = n_dur > 1 ? (double)j / (double)(n_dur - 1) : 0.0;
    out[idx] = exp(log(q_lo) * (1.0 - x) + log(q_hi) * x);
}

}  // namespace

void launch_period_grid(double a3, double c, long long n_per, double* out, cudaStream_t st) {
    k_period_grid<<<(unsigned)((n_per + 255) / 256), 256, 0, st>>>(a3, c, n_per, out);
}

void launch_duration_grid(const double* periods, long long n_per, int n_dur, double k_min, double k_max,
                          double q_cap, double* out, int* bad, cudaStream_t st) {
    const long long total = n_per * n_dur;
    k_duration_grid<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(periods, n_per, n_dur, k_min, k_max, q_cap, out, bad);
}

}  // namespace gtls
