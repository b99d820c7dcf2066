// mppi_peaks.cu -- roofline denominators measured on the device in use:
// an FFMA-throughput loop for the FP32 ALU peak and a device-to-device copy for HBM bandwidth.
// MEASURED_PEAKS.json has no FP32 entry, so the rollout's "alu" roofline needs this number.
#include <algorithm>
#include <cuda_runtime.h>

#include "../../include/mppi.h"

namespace {

// 16 independent FMA chains per thread: enough ILP to saturate both FMA pipes of a scheduler.
__global__ void __launch_bounds__(256) fma_peak_kernel(float* out, int iters, float a, float b)
{
    float v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = a + (float)(threadIdx.x + i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int i = 0; i < 16; ++i) v[i] = fmaf(v[i], a, b);
    }
    float s = 0.0f;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += v[i];
    if (s == 123.456f) out[0] = s;    // never true: keeps the loop alive
}

__global__ void __launch_bounds__(256) copy_kernel(const float4* __restrict__ src, float4* __restrict__ dst, size_t n)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) dst[i] = __ldcs(src + i);
}

}  // namespace

extern "C" int mppi_measure_fma_peak(int reps, double* tflops, double* sm_clock_mhz)
{
    if (!tflops) return MPPI_E_NULL;
    int dev = 0, sms = 0, khz = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return MPPI_E_CUDA;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev);
    float* d = nullptr;
    if (cudaMalloc(&d, 256) != cudaSuccess) return MPPI_E_ALLOC;
    const int iters = 4096, blocks = sms * 8, threads = 256;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = 0.0;
    for (int r = 0; r < std::max(reps, 1) + 1; ++r) {
        cudaEventRecord(e0);
        fma_peak_kernel<<<blocks, threads>>>(d, iters, 1.0000001f, 1e-9f);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(d); return MPPI_E_CUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flops = 2.0 * 16 * 8 * (double)iters * threads * blocks;
        if (r > 0) best = std::max(best, flops / (ms * 1e-3) / 1e12);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
    *tflops = best;
    if (sm_clock_mhz) *sm_clock_mhz = khz / 1000.0;
    return cudaGetLastError() == cudaSuccess ? MPPI_OK : MPPI_E_CUDA;
}

extern "C" int mppi_measure_copy_bw(int64_t bytes, int reps, double* gbs)
{
    if (!gbs) return MPPI_E_NULL;
    if (bytes < 16) return MPPI_E_RANGE;
    const size_t n = (size_t)bytes / 16;
    float4 *a = nullptr, *b = nullptr;
    if (cudaMalloc(&a, n * 16) != cudaSuccess) return MPPI_E_ALLOC;
    if (cudaMalloc(&b, n * 16) != cudaSuccess) { cudaFree(a); return MPPI_E_ALLOC; }
    cudaMemset(a, 1, n * 16);
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = 0.0;
    for (int r = 0; r < std::max(reps, 1) + 1; ++r) {
        cudaEventRecord(e0);
        copy_kernel<<<sms * 16, 256>>>(a, b, n);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(a); cudaFree(b); return MPPI_E_CUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0) best = std::max(best, 2.0 * n * 16 / (ms * 1e-3) / 1e9);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(a); cudaFree(b);
    *gbs = best;
    return cudaGetLastError() == cudaSuccess ? MPPI_OK : MPPI_E_CUDA;
}
