// mppi_scan.cu -- instantiation and launch of the time-parallel latency kernel (mppi_scan.cuh).
#include <cstring>
#include "mppi_internal.h"
#include "mppi_scan.cuh"

namespace mppi {

typedef void (*ScanFn)(const DevParams, const StepArgs);

template <int OBJ>
static ScanFn pick_scan1(const LaunchCfg& c)
{
    if (c.fast_math) return c.store_du ? rollout_scan_kernel<OBJ, 1, true> : rollout_scan_kernel<OBJ, 1, false>;
    return c.store_du ? rollout_scan_kernel<OBJ, 0, true> : rollout_scan_kernel<OBJ, 0, false>;
}
static ScanFn pick_scan(const LaunchCfg& c)
{
    return c.objective == OBJ_GATE_PAPER ? pick_scan1<OBJ_GATE_PAPER>(c) : pick_scan1<OBJ_GATE>(c);
}

size_t scan_smem_bytes(const DevParams& P, const LaunchCfg& c)
{
    return ((size_t)P.N + track_f4(P, c.objective) + 16 + scan_extra_f4(P.N, P.blocks_per_ctrl, c.scan)) * sizeof(float4);
}

const void* scan_kernel_ptr(const LaunchCfg& c) { return reinterpret_cast<const void*>(pick_scan(c)); }

cudaError_t launch_scan(const DevParams& P, const StepArgs& A, const LaunchCfg& c, cudaStream_t s, bool pdl)
{
    const dim3 grid(P.blocks_per_ctrl, P.B), block(c.block_threads);
    if (pdl) {
        // programmatic dependent launch (StepArgs::pdl bit 0 must be set): see launch_rollout
        cudaLaunchConfig_t lc;
        memset(&lc, 0, sizeof lc);
        lc.gridDim = grid; lc.blockDim = block; lc.dynamicSmemBytes = c.smem_bytes; lc.stream = s;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        lc.attrs = at; lc.numAttrs = 1;
        return cudaLaunchKernelEx(&lc, pick_scan(c), P, A);
    }
    pick_scan(c)<<<grid, block, c.smem_bytes, s>>>(P, A);
    return cudaGetLastError();
}

}  // namespace mppi
