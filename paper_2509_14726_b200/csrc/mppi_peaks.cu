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

// ---------------------------------------------------------------------------------------------
// Issue rates of the instruction classes the rollout loop is made of ("Ceiling of this
// instruction mix"): cycles per warp-instruction per SM sub-partition at saturation (8 resident warps per
// sub-partition, 8 independent chains per thread), measured with clock64 inside the kernel.  The operands are
// loaded from memory so that the compiler cannot fold them into immediates or the constant bank.
//   0 FFMA  three distinct register operands        1 FFMA  one constant / uniform-register operand
//   2 FFMA2 (fma.rn.f32x2) three register pairs     3 FMUL  reg, reg          4 FADD reg, reg
//   5 IMAD.WIDE.U32 + LOP3 (one Philox half-round: two instructions)
//   6 MUFU.EX2                                      7 FMNMX reg, reg
// ---------------------------------------------------------------------------------------------
namespace {

constexpr int kRateClasses = 8;
constexpr int kRateChains = 8, kRateInner = 16;     // 8 warps per sub-partition x 8 chains in flight

template <int CLS>
__global__ void __launch_bounds__(1024, 1) rate_kernel(const float* __restrict__ in, float* out, long long* cycles, int iters, float kc)
{
    // every chain has operands of its own (x_i, y_i): consecutive instructions share no register, so the operand
    // reuse cache cannot hide the register-file reads the rollout's FFMAs really make
    float v[kRateChains], x[kRateChains], y[kRateChains];
    unsigned int u[kRateChains];
#pragma unroll
    for (int i = 0; i < kRateChains; ++i) {
        x[i] = in[0] + 1e-7f * (float)(i + (threadIdx.x & 3)); y[i] = in[1] * (float)(i + 1 + (threadIdx.x & 1));   // per-thread: not uniform registers
        v[i] = in[2] + (float)(threadIdx.x + i); u[i] = __float_as_uint(v[i]);
    }
    unsigned long long p[kRateChains / 2], px[kRateChains / 2], py[kRateChains / 2];
#pragma unroll
    for (int i = 0; i < kRateChains / 2; ++i) {
        p[i] = ((unsigned long long)__float_as_uint(v[2 * i]) << 32) | __float_as_uint(v[2 * i + 1]);
        px[i] = ((unsigned long long)__float_as_uint(x[2 * i]) << 32) | __float_as_uint(x[2 * i + 1]);
        py[i] = ((unsigned long long)__float_as_uint(y[2 * i]) << 32) | __float_as_uint(y[2 * i + 1]);
    }
    __syncthreads();
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < kRateInner; ++r) {
            if (CLS == 2) {
#pragma unroll
                for (int i = 0; i < kRateChains / 2; ++i)
                    asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(p[i]) : "l"(px[i]), "l"(py[i]));
            } else {
#pragma unroll
                for (int i = 0; i < kRateChains; ++i) {
                    if (CLS == 0) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(v[i]) : "f"(x[i]), "f"(y[i]));
                    if (CLS == 1) v[i] = fmaf(v[i], kc, y[i]);
                    if (CLS == 3) asm volatile("mul.rn.f32 %0, %0, %1;" : "+f"(v[i]) : "f"(x[i]));
                    if (CLS == 4) asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(v[i]) : "f"(y[i]));
                    if (CLS == 5) {
                        unsigned int lo, hi;
                        asm volatile("mul.lo.u32 %0, %2, 0xD2511F53;\n\tmul.hi.u32 %1, %2, 0xD2511F53;" : "=r"(lo), "=r"(hi) : "r"(u[i]));
                        u[i] = hi ^ lo ^ (unsigned int)it;
                    }
                    if (CLS == 6) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(v[i]));
                    if (CLS == 7) asm volatile("min.f32 %0, %0, %1;" : "+f"(v[i]) : "f"(x[i]));
                }
            }
        }
    }
    const long long t1 = clock64();
    float s = 0.0f;
#pragma unroll
    for (int i = 0; i < kRateChains; ++i) s += v[i] + __uint_as_float(u[i]);
#pragma unroll
    for (int i = 0; i < kRateChains / 2; ++i) s += __uint_as_float((unsigned int)p[i]) + __uint_as_float((unsigned int)(p[i] >> 32));
    if (s == 123.456f) out[0] = s;                    // never true: keeps the loops alive
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

template <int CLS>
int run_rate(int sms, const float* d_in, float* d_out, long long* d_cyc, double* cyc_per_instr)
{
    // one block of 1024 threads per SM: exactly 8 resident warps per sub-partition, whatever the register count
    const int blocks = sms, iters = 512;
    rate_kernel<CLS><<<blocks, 1024>>>(d_in, d_out, d_cyc, 8, 1.0000001f);       // warm-up
    rate_kernel<CLS><<<blocks, 1024>>>(d_in, d_out, d_cyc, iters, 1.0000001f);
    if (cudaDeviceSynchronize() != cudaSuccess) return MPPI_E_CUDA;
    long long* h = new long long[blocks];
    cudaMemcpy(h, d_cyc, sizeof(long long) * blocks, cudaMemcpyDeviceToHost);
    std::sort(h, h + blocks);
    const double cyc = (double)h[blocks / 2];
    delete[] h;
    // per sub-partition: 32 warps / 4 sub-partitions = 8 warps, each issuing iters x inner x n instructions
    const double per_warp = (double)iters * kRateInner * (CLS == 2 ? kRateChains / 2 : kRateChains);
    *cyc_per_instr = cyc / (8.0 * per_warp);
    return MPPI_OK;
}

}  // namespace

extern "C" int mppi_measure_issue_rates(double* cycles_per_instr, int n)
{
    if (!cycles_per_instr) return MPPI_E_NULL;
    if (n < kRateClasses) return MPPI_E_RANGE;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return MPPI_E_CUDA;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    float* d_in = nullptr; float* d_out = nullptr; long long* d_cyc = nullptr;
    if (cudaMalloc(&d_in, 64) != cudaSuccess || cudaMalloc(&d_out, 64) != cudaSuccess ||
        cudaMalloc(&d_cyc, sizeof(long long) * sms) != cudaSuccess) {
        cudaFree(d_in); cudaFree(d_out); cudaFree(d_cyc);
        return MPPI_E_ALLOC;
    }
    const float h_in[4] = {1.0000001f, 1e-9f, 0.5f, 0.0f};
    cudaMemcpy(d_in, h_in, sizeof h_in, cudaMemcpyHostToDevice);
    int rc = MPPI_OK;
    if (rc == MPPI_OK) rc = run_rate<0>(sms, d_in, d_out, d_cyc, cycles_per_instr + 0);
    if (rc == MPPI_OK) rc = run_rate<1>(sms, d_in, d_out, d_cyc, cycles_per_instr + 1);
    if (rc == MPPI_OK) rc = run_rate<2>(sms, d_in, d_out, d_cyc, cycles_per_instr + 2);
    if (rc == MPPI_OK) rc = run_rate<3>(sms, d_in, d_out, d_cyc, cycles_per_instr + 3);
    if (rc == MPPI_OK) rc = run_rate<4>(sms, d_in, d_out, d_cyc, cycles_per_instr + 4);
    if (rc == MPPI_OK) rc = run_rate<5>(sms, d_in, d_out, d_cyc, cycles_per_instr + 5);
    if (rc == MPPI_OK) rc = run_rate<6>(sms, d_in, d_out, d_cyc, cycles_per_instr + 6);
    if (rc == MPPI_OK) rc = run_rate<7>(sms, d_in, d_out, d_cyc, cycles_per_instr + 7);
    cudaFree(d_in); cudaFree(d_out); cudaFree(d_cyc);
    return rc;
}

// ---------------------------------------------------------------------------------------------
// What a CUDA-event pair around ANY kernel launch costs on this device: an empty kernel of the lone-controller
// grid (128 blocks x 256 threads), each launch behind a kernel that keeps the GPU busy so that the host runs ahead
// as in bench.py's timed loop.  Context for the iteration latency: this much of it is not the library's.
// ---------------------------------------------------------------------------------------------
namespace {
__global__ void empty_kernel(int* p) { if (p && threadIdx.x == 9999) *p = 0; }
__global__ void busy_kernel(float* p, int n)
{
    float v = (float)threadIdx.x;
    for (int i = 0; i < n; ++i) v = fmaf(v, 1.0000001f, 1e-9f);
    if (v == 123.456f) *p = v;
}
}  // namespace

extern "C" int mppi_measure_launch_floor(int reps, double* median_us)
{
    if (!median_us) return MPPI_E_NULL;
    reps = std::min(std::max(reps, 8), 4096);
    float* d = nullptr;
    if (cudaMalloc(&d, 64) != cudaSuccess) return MPPI_E_ALLOC;
    cudaEvent_t* ev = new cudaEvent_t[2 * reps];
    for (int i = 0; i < 2 * reps; ++i) cudaEventCreate(&ev[i]);
    for (int i = 0; i < reps; ++i) {
        busy_kernel<<<148, 256>>>(d, 20000);                     // ~ 40 us: the host queues ahead of the device
        cudaEventRecord(ev[2 * i]);
        empty_kernel<<<128, 256>>>(nullptr);
        cudaEventRecord(ev[2 * i + 1]);
    }
    int rc = cudaDeviceSynchronize() == cudaSuccess ? MPPI_OK : MPPI_E_CUDA;
    float* ms = new float[reps];
    for (int i = 0; i < reps && rc == MPPI_OK; ++i) cudaEventElapsedTime(&ms[i], ev[2 * i], ev[2 * i + 1]);
    if (rc == MPPI_OK) {
        std::sort(ms, ms + reps);
        *median_us = 1e3 * ms[reps / 2];
    }
    for (int i = 0; i < 2 * reps; ++i) cudaEventDestroy(ev[i]);
    delete[] ev; delete[] ms; cudaFree(d);
    return rc;
}
