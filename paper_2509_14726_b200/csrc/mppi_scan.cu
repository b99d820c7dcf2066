// mppi_scan.cu -- instantiation and launch of the time-parallel latency kernel (mppi_scan.cuh).
#include "mppi_internal.h"
#include "mppi_scan.cuh"

namespace mppi {

typedef void (*ScanFn)(const DevParams, const StepArgs);

static ScanFn pick_scan(const LaunchCfg& c)
{
    if (c.fast_math) return c.store_du ? rollout_scan_kernel<OBJ_GATE, 1, true> : rollout_scan_kernel<OBJ_GATE, 1, false>;
    return c.store_du ? rollout_scan_kernel<OBJ_GATE, 0, true> : rollout_scan_kernel<OBJ_GATE, 0, false>;
}

size_t scan_smem_bytes(const DevParams& P, const LaunchCfg& c)
{
    return ((size_t)P.N + track_f4(P, c.objective) + 16 + scan_extra_f4(P.N, P.blocks_per_ctrl)) * sizeof(float4);
}

const void* scan_kernel_ptr(const LaunchCfg& c) { return reinterpret_cast<const void*>(pick_scan(c)); }

cudaError_t launch_scan(const DevParams& P, const StepArgs& A, const LaunchCfg& c, cudaStream_t s)
{
    pick_scan(c)<<<dim3(P.blocks_per_ctrl, P.B), kScanThreads, c.smem_bytes, s>>>(P, A);
    return cudaGetLastError();
}

}  // namespace mppi
