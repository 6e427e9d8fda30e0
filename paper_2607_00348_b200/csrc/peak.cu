// FP64 pipe microbenchmark: the roofline denominator of the in-transit chi2 stage (bench.py --peak-fp64).
// Nothing of the search runs here.  Every thread keeps 16 independent accumulators a_i = fma(b_i, c_i, a_i)
// with three distinct register operands per DFMA (the operand pattern of the ring kernels), four warps per
// SM sub-partition, no memory traffic inside the timed loop.  The derived peak it is compared with is
// 148 SMs x 64 DFMA lanes/clk x 2 flop x SM clock.
#include "gtls_internal.cuh"

namespace gtls {
namespace {

constexpr int kPeakChains = 16;
constexpr int kPeakInner = 8;      // unrolled rounds per loop trip

__global__ void __launch_bounds__(128) k_peak_fp64(double* out, const double* __restrict__ seed, int trips) {
    double a[kPeakChains], b[kPeakChains], c[kPeakChains];
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) {
        a[i] = seed[i] + threadIdx.x;
        b[i] = seed[kPeakChains + i] * (1.0 + threadIdx.x);
        c[i] = seed[2 * kPeakChains + i];
    }
#pragma unroll 1
    for (int t = 0; t < trips; ++t) {
#pragma unroll
        for (int r = 0; r < kPeakInner; ++r)
#pragma unroll
            for (int i = 0; i < kPeakChains; ++i) a[i] = fma(b[i], c[i], a[i]);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) s += a[i];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace
}  // namespace gtls

using namespace gtls;

extern "C" int gtls_peak_fp64(double seconds, const gtls_opts* opts, double* out_tflops, double* out_ms,
                              int64_t* out_launches) {
    if (!(seconds > 0.0) || seconds > 60.0 || !out_tflops) return GTLS_EINVAL;
    const int device = opts ? opts->device : 0;
    cudaStream_t st = opts ? (cudaStream_t)opts->stream : nullptr;
    if (cudaSetDevice(device) != cudaSuccess) return GTLS_ECUDA;
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) return GTLS_ECUDA;
    const int grid = sms * 4, threads = 128;          // 16 warps per SM = 4 per sub-partition
    double* d = nullptr;
    if (cudaMalloc((void**)&d, ((size_t)grid * threads + 3 * kPeakChains) * sizeof(double)) != cudaSuccess) return GTLS_ENOMEM;
    double h[3 * kPeakChains];
    for (int i = 0; i < kPeakChains; ++i) { h[i] = 1.0 + i; h[kPeakChains + i] = 1e-9 * (i + 1); h[2 * kPeakChains + i] = 1.0 + 1e-9 * i; }
    double* seed = d + (size_t)grid * threads;
    cudaMemcpyAsync(seed, h, sizeof(h), cudaMemcpyHostToDevice, st);
    const int trips = 4000;                           // ~2 ms per launch
    const double flop_per_launch = 2.0 * kPeakChains * kPeakInner * (double)trips * threads * grid;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    k_peak_fp64<<<grid, threads, 0, st>>>(d, seed, trips);          // warm-up
    cudaStreamSynchronize(st);
    // launches back to back on the stream until `seconds` of device time have gone by
    double total_ms = 0.0;
    int64_t launches = 0;
    int rc = GTLS_OK;
    while (total_ms < seconds * 1e3) {
        const int burst = 8;
        cudaEventRecord(e0, st);
        for (int k = 0; k < burst; ++k) k_peak_fp64<<<grid, threads, 0, st>>>(d, seed, trips);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { rc = GTLS_ECUDA; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        total_ms += ms; launches += burst;
    }
    if (cudaGetLastError() != cudaSuccess) rc = GTLS_ECUDA;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(d);
    if (rc != GTLS_OK) return rc;
    *out_tflops = flop_per_launch * (double)launches / (total_ms * 1e-3) / 1e12;
    if (out_ms) *out_ms = total_ms;
    if (out_launches) *out_launches = launches;
    return GTLS_OK;
}
