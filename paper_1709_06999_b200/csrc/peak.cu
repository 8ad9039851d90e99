// peak.cu — gal_measure_fp64_fma_peak: the FP64 fused-multiply-add rate this GPU sustains, measured, so that the
// ALU fractions bench.py reports ("measures an FP64 FMA peak on the box and reports both fractions per
// kernel") rest on a number taken on the box instead of on unit counts x nominal clock.  Not on the hot path.
//
// Eight independent DFMA chains per thread (the FP64 pipe's latency is covered many times over by 64 resident warps
// per SM x 8 chains), 8 CTAs of 256 threads per SM, a few milliseconds per launch, CUDA events around each launch,
// best of five after a warm-up launch.
#include "../../include/galario_b200.h"

#include <cuda_runtime.h>

namespace {

constexpr int PEAK_CHAINS = 8;
constexpr int PEAK_ITERS = 1 << 14;

__global__ void __launch_bounds__(256) fp64_fma_peak_kernel(double* out, double a, double b) {
    double x[PEAK_CHAINS];
#pragma unroll
    for (int j = 0; j < PEAK_CHAINS; ++j) x[j] = 1.0 + 1e-3 * (double)(threadIdx.x + j);
#pragma unroll 1
    for (int i = 0; i < PEAK_ITERS; i += 4) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int j = 0; j < PEAK_CHAINS; ++j) x[j] = fma(x[j], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int j = 0; j < PEAK_CHAINS; ++j) s += x[j];
    if (s == 123.456) *out = s;                              // (never true: keeps the chains alive)
}

}  // namespace

extern "C" int gal_measure_fp64_fma_peak(int device, double* tflops_out, double* ms_out) {
    if (device < 0 || !tflops_out) return GAL_ERR_INVALID_ARGUMENT;
    int prev = -1, sms = 0;
    if (cudaGetDevice(&prev) != cudaSuccess || cudaSetDevice(device) != cudaSuccess) return GAL_ERR_CUDA;
    int rc = GAL_ERR_CUDA;
    double* out = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    float best = 1e30f;
    do {
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) break;
        if (cudaMalloc((void**)&out, sizeof(double)) != cudaSuccess) { rc = GAL_ERR_ALLOC; break; }
        if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) break;
        const unsigned grid = (unsigned)sms * 8u;
        bool ok = true;
        for (int rep = 0; rep < 6 && ok; ++rep) {            // rep 0 warms up
            ok = cudaEventRecord(e0, 0) == cudaSuccess;
            fp64_fma_peak_kernel<<<grid, 256>>>(out, 0.999999, 1e-6);
            ok = ok && cudaGetLastError() == cudaSuccess && cudaEventRecord(e1, 0) == cudaSuccess &&
                 cudaEventSynchronize(e1) == cudaSuccess;
            float ms = 0.f;
            ok = ok && cudaEventElapsedTime(&ms, e0, e1) == cudaSuccess;
            if (ok && rep > 0 && ms < best) best = ms;
        }
        if (!ok) break;
        const double flops = 2.0 * (double)grid * 256.0 * PEAK_CHAINS * (double)PEAK_ITERS;
        *tflops_out = flops / ((double)best * 1e-3) / 1e12;
        if (ms_out) *ms_out = (double)best;
        rc = GAL_OK;
    } while (false);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (out) cudaFree(out);
    if (prev != device) cudaSetDevice(prev);
    return rc;
}
