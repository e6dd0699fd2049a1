// fma_peak.cu -- register-resident FMA chain microbenchmark: the measured ALU roofline
// denominator (SURVEY 8(d) "Peaks": >= 8 independent accumulators per thread, full occupancy,
// back to back for `seconds`, sustained TFLOP/s).
#include "common.cuh"

namespace tkhp {

template <typename real>
__global__ void __launch_bounds__(256) k_fma_chain(real *out, int iters, real a, real b) {
    real x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            x0 = x0 * a + b; x1 = x1 * a + b; x2 = x2 * a + b; x3 = x3 * a + b;
            x4 = x4 * a + b; x5 = x5 * a + b; x6 = x6 * a + b; x7 = x7 * a + b;
        }
    }
    real s = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
    if (s == (real)123456.789) out[0] = s;   // never true: keeps the chain alive
}

// the caller's current device is put back on every return path
struct PeakDeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit PeakDeviceGuard(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        ok = cudaSetDevice(dev) == cudaSuccess;
    }
    ~PeakDeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

template <typename real>
static int run_peak(int device, double seconds, double *tflops) {
    cudaDeviceProp prop;
    PeakDeviceGuard guard(device);
    if (!guard.ok || cudaGetDeviceProperties(&prop, device) != cudaSuccess) { cudaGetLastError(); return TKHP_ECUDA; }
    real *out = nullptr;   // one scalar the chain never writes (this benchmark call allocates; see tkhp.h)
    if (cudaMalloc(&out, sizeof(real)) != cudaSuccess) return TKHP_ECUDA;
    const int ctas = prop.multiProcessorCount * 8;   // 8 x 256 threads = 2048 threads per SM
    const int iters = 4096;
    const double flops_per_launch = 2.0 * 8 * 16 * (double)iters * 256.0 * ctas;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    k_fma_chain<real><<<ctas, 256>>>(out, iters, (real)0.999, (real)0.001);   // warm-up
    cudaDeviceSynchronize();
    double best_window = 0.0, elapsed = 0.0, total_flops = 0.0;
    while (elapsed < seconds) {
        cudaEventRecord(e0);
        for (int r = 0; r < 8; ++r) k_fma_chain<real><<<ctas, 256>>>(out, iters, (real)0.999, (real)0.001);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) {
            cudaEventDestroy(e0); cudaEventDestroy(e1);
            cudaFree(out);
            return TKHP_ECUDA;
        }
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        elapsed += ms * 1e-3;
        total_flops += 8 * flops_per_launch;
        double w = 8 * flops_per_launch / (ms * 1e-3);
        if (w > best_window) best_window = w;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    *tflops = total_flops / elapsed * 1e-12;   // sustained over the whole run
    return TKHP_OK;
}

}  // namespace tkhp

extern "C" int tkhp_fma_peak(int32_t device, int32_t precision, double seconds, double *tflops) {
    if (!tflops || seconds <= 0.0) return TKHP_EINVAL;
    if (precision == TKHP_MIXED || precision == TKHP_FIXED) return tkhp::run_peak<float>(device, seconds, tflops);
    if (precision == TKHP_FP64) return tkhp::run_peak<double>(device, seconds, tflops);
    return TKHP_EINVAL;
}
