// mppi_rate.cu -- the rollout under the paper's OWN input model: the control input is
// the thrust RATE u = dT/dt and the four rotor thrusts are states ("Following the approach
// in [4] ..."), with the rate and thrust ranges of Table I, the rotor-drag term
// - R D R^T v of eq.(2) and a soft body-rate limit ("external cost").
// Readings R-27..R-32 of DESIGN.md.  First correct path: one sample per thread, the 17-dim state in
// registers, a general 4-stage RK4 (the drag makes v' depend on v, so the triangular short-cuts of
// rk4_step do not apply), the same objectives and the same fused softmax update as rollout_kernel.
#include "mppi_internal.h"
#include "mppi_rollout.cuh"
#include "mppi_rate.cuh"
#include "mppi_pipe_rate.cuh"

namespace mppi {

// grid = (K / blockDim.x, B), one sample per thread; shared-memory carve-up as rollout_kernel
template <int OBJ, int MATH, bool STORE_DU, bool FUSED>
__global__ void __launch_bounds__(256, 3) rollout_rate_kernel(const DevParams P, const StepArgs A)
{
    extern __shared__ float4 smem[];
    const int tid = threadIdx.x;
    const int b = blockIdx.y;
    const int k = blockIdx.x * blockDim.x + tid;
    const int N = P.N;

    float4* s_unom = smem;
    float4* s_trk = smem + N;
    float* s_red = reinterpret_cast<float*>(s_trk + track_f4(P, OBJ));   // 64 floats
    float4* s_acc = reinterpret_cast<float4*>(s_red + 64);
    float* s_pair = reinterpret_cast<float*>(s_acc + (blockDim.x >> 5) * N);
    // OBJ_CONTOUR_PAPER: nominal of the fifth input [N] + one accumulator row per warp, after the pair area
    float* s_vnom = s_pair + 4 * ((3 * P.blocks_per_ctrl + 3) / 4);
    float* s_acc5 = s_vnom + N;

    const int start = A.start[b];
    stage_inputs<OBJ>(P, A, b, start, s_unom, s_trk);
    if (OBJ == OBJ_CONTOUR_PAPER)
        for (int t = tid; t < N; t += blockDim.x) s_vnom[t] = A.v_nom[(size_t)b * N + t];
    __syncthreads();

    const float* xb = A.x0 + (OBJ == OBJ_CONTOUR_PAPER ? 19 : 17) * b;   // p, q, v, omega, T(4) [, theta, v_theta]
    State x = load_state(xb);
    float4 T = make_float4(xb[13], xb[14], xb[15], xb[16]);
    float theta = 0.0f, v_theta = 0.0f;                                  // OBJ_CONTOUR_PAPER: progress states [R-33]
    if (OBJ == OBJ_CONTOUR_PAPER) { theta = xb[17]; v_theta = xb[18]; }
    const int i0 = OBJ == OBJ_CONTOUR ? contour_start_index(P, s_trk, start, x, s_red) : 0;
    const float lo = -P.rate_max, hi = P.rate_max;                       // [R-28]

    float J = 0.0f;
    GateCost gc;
    GatePaperCost gp;
    ContourCost cc;
    const int* s_front = reinterpret_cast<const int*>(s_trk + 4 * P.G);  // OBJ_GATE_PAPER only
    if (OBJ == OBJ_GATE) gc.init<MATH>(P, s_trk, start, x);
    if (OBJ == OBJ_GATE_PAPER) gp.init(P, s_trk, start, x);
    if (OBJ == OBJ_CONTOUR) cc.init(P, s_trk, i0, x);
    float4* du_out = STORE_DU ? A.du + (size_t)b * N * P.K + k : nullptr;
    for (int t = 0; t < N; ++t) {
        const float4 un = s_unom[t];
        const float4 u = sample_input<MATH>(P, A.rk, (uint32_t)k, (uint32_t)t, A.iter, (uint32_t)b, un, lo, hi);
        if (STORE_DU) du_out[(size_t)t * P.K] = make_float4(u.x - un.x, u.y - un.y, u.z - un.z, u.w - un.w);
        if (OBJ == OBJ_TRACK)      // eq.(8): the input term acts on the inputs = the rates [R-32]
            J += fmaf(P.R, u.x * u.x + u.y * u.y + u.z * u.z + u.w * u.w, track_state_term(P, s_trk + 4 * t, x));
        if (OBJ == OBJ_CONTOUR_PAPER) {            // fifth sampled input, stage cost, progress states [R-34]..[R-37]
            const float dv = sample_progress_accel<MATH>(P, A.rk, (uint32_t)k, (uint32_t)t, A.iter, (uint32_t)b,
                                                         s_vnom[t]);
            J += contour_paper_stage(P, s_trk, x, theta, v_theta, u, dv);
            theta = fmaf(P.hh2, dv, fmaf(P.dt, v_theta, theta));
            v_theta = fminf(fmaxf(fmaf(P.dt, dv, v_theta), 0.0f), P.v_theta_max);
        }
        rk4_rate_step(P, x, T, u);
        J += rate_limit_cost(P, x);
        if (OBJ == OBJ_GATE) gc.step<MATH>(P, s_trk, x);
        if (OBJ == OBJ_GATE_PAPER) gp.step(P, s_trk, s_front, x, t);
        if (OBJ == OBJ_CONTOUR) J += cc.step(P, s_trk, x);
    }
    if (OBJ == OBJ_GATE) J += gc.finish<MATH>(P, s_trk, x);
    if (OBJ == OBJ_GATE_PAPER) J += gp.finish(P);
    if (OBJ == OBJ_TRACK) J += track_state_term(P, s_trk + 4 * N, x);
    A.cost[(size_t)b * P.K + k] = J;

    if (!FUSED) return;
    if (OBJ == OBJ_CONTOUR_PAPER)
        block_partial_and_combine<MATH>(P, A, b, blockIdx.x, J, lo, hi, s_unom, s_red, s_acc, s_pair, s_vnom, s_acc5);
    else
        block_partial_and_combine<MATH>(P, A, b, blockIdx.x, J, lo, hi, s_unom, s_red, s_acc, s_pair);
}

// ---- host-side dispatch ------------------------------------------------------------------------------
typedef void (*RateFn)(const DevParams, const StepArgs);

template <int OBJ, int MATH>
static RateFn pick_rate2(const LaunchCfg& c)
{
    if (c.fused) return c.store_du ? rollout_rate_kernel<OBJ, MATH, true, true> : rollout_rate_kernel<OBJ, MATH, false, true>;
    return rollout_rate_kernel<OBJ, MATH, true, false>;
}
template <int OBJ>
static RateFn pick_rate1(const LaunchCfg& c)
{
    return c.fast_math ? pick_rate2<OBJ, 1>(c) : pick_rate2<OBJ, 0>(c);
}
static RateFn pick_rate(const LaunchCfg& c)
{
    switch (c.objective) {
        case OBJ_GATE: return pick_rate1<OBJ_GATE>(c);
        case OBJ_GATE_PAPER: return pick_rate1<OBJ_GATE_PAPER>(c);
        case OBJ_TRACK: return pick_rate1<OBJ_TRACK>(c);
        case OBJ_CONTOUR_PAPER: return pick_rate1<OBJ_CONTOUR_PAPER>(c);
        default: return pick_rate1<OBJ_CONTOUR>(c);
    }
}

template <int OBJ, bool SHALLOW>
static RateFn pick_pipe_rate2(const LaunchCfg& c)
{
    if (c.fast_math) return c.store_du ? rollout_pipe_rate_kernel<OBJ, 1, true, SHALLOW> : rollout_pipe_rate_kernel<OBJ, 1, false, SHALLOW>;
    return c.store_du ? rollout_pipe_rate_kernel<OBJ, 0, true, SHALLOW> : rollout_pipe_rate_kernel<OBJ, 0, false, SHALLOW>;
}
template <int OBJ>
static RateFn pick_pipe_rate1(const LaunchCfg& c)
{
    return c.pipe_shallow ? pick_pipe_rate2<OBJ, true>(c) : pick_pipe_rate2<OBJ, false>(c);
}
static RateFn pick_pipe_rate(const LaunchCfg& c)
{
    switch (c.objective) {
        case OBJ_GATE: return pick_pipe_rate1<OBJ_GATE>(c);
        case OBJ_GATE_PAPER: return pick_pipe_rate1<OBJ_GATE_PAPER>(c);
        case OBJ_CONTOUR_PAPER: return pick_pipe_rate1<OBJ_CONTOUR_PAPER>(c);
        default: return pick_pipe_rate1<OBJ_TRACK>(c);
    }
}

const void* rate_kernel_ptr(const LaunchCfg& c)
{
    return reinterpret_cast<const void*>(c.pipe ? pick_pipe_rate(c) : pick_rate(c));
}

cudaError_t launch_rate(const DevParams& P, const StepArgs& A, const LaunchCfg& c, cudaStream_t s)
{
    (c.pipe ? pick_pipe_rate(c) : pick_rate(c))<<<dim3(P.blocks_per_ctrl, P.B), c.block_threads, c.smem_bytes, s>>>(P, A);
    return cudaGetLastError();
}

}  // namespace mppi
