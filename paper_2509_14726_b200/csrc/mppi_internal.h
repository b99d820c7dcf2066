// mppi_internal.h -- host-side declarations shared by mppi_api.cu and mppi_kernels.cu.
#pragma once
#include "mppi_device.cuh"

namespace mppi {

struct LaunchCfg {
    int objective;      // OBJ_*
    int fast_math;      // 0 / 1
    int store_du;       // 0 / 1
    int fused;          // 1: MPPI_PIPE_FUSED, 0: MPPI_PIPE_TWO_PASS
    int block_threads;  // rollout block size
    int packed;         // 1: rollout2_kernel, two samples per thread in fp32x2 registers
    int pipe;           // 1: rollout_pipe_kernel, one rollout pipelined over three warps (32 samples per block)
    int rate;           // 1: rollout_rate_kernel (thrust-rate input model, mppi_rate.cu)
    int pipe_shallow;   // rollout_pipe_rate_kernel: 1 = rings (2, 2) chunks deep (two blocks per SM), 0 = (4, 3)
    int lat_consumers;  // 0: throughput kernel; 1, 2 or 4: latency kernel with that many rollout warps per block
    int lat_split;      // latency kernel, search-contouring: 1 = the search runs in warps of its own (when it fits in shared memory)
    int scan;           // > 0: rollout_scan_kernel, one rollout split over 16 lanes along the horizon (mppi_scan.cuh);
                        // the value is the number of samples per block (even, 8..32); block_threads = 16 x that
    size_t smem_bytes;  // dynamic shared memory of the rollout kernel
};

// dynamic shared memory the rollout kernel needs for this configuration
size_t rollout_smem_bytes(const DevParams& P, const LaunchCfg& c);

// kernel function pointers (for cudaFuncGetAttributes / graph nodes)
const void* rollout_kernel_ptr(const LaunchCfg& c);
const void* reduce_kernel_ptr();
const void* sim_kernel_ptr();

cudaError_t launch_rollout(const DevParams& P, const StepArgs& A, const LaunchCfg& c, cudaStream_t s, bool pdl = false);
cudaError_t launch_reduce(const DevParams& P, const StepArgs& A, cudaStream_t s);
cudaError_t launch_sim_progress(const DevParams& P, float* x, const float* u_new, float* u_nom_next,
                                const float* v_new, float* v_nom_next, cudaStream_t s);
cudaError_t launch_sim(const DevParams& P, int objective, float* x, int* start, const float* u_new,
                       float* u_nom_next, cudaStream_t s);

// mppi_rate.cu: the thrust-rate input model
const void* rate_kernel_ptr(const LaunchCfg& c);
cudaError_t launch_rate(const DevParams& P, const StepArgs& A, const LaunchCfg& c, cudaStream_t s);

// mppi_scan.cu: the time-parallel latency kernel
const void* scan_kernel_ptr(const LaunchCfg& c);
cudaError_t launch_scan(const DevParams& P, const StepArgs& A, const LaunchCfg& c, cudaStream_t s, bool pdl = false);
size_t scan_smem_bytes(const DevParams& P, const LaunchCfg& c);

cudaError_t launch_front(const DevParams& P, const float* x0, const int* start, const float* u, int* front,
                         cudaStream_t s);

constexpr int kReduceThreads = 256;

}  // namespace mppi
