// mppi_rate.cu -- the rollout under the paper's OWN input model: the control input is
// the thrust RATE u = dT/dt and the four rotor thrusts are states ("Following the approach
// in [4] ..."), with the rate and thrust ranges of Table I, the rotor-drag term
// - R D R^T v of eq.(2) and a soft body-rate limit ("external cost").
// Readings R-27..R-32 of DESIGN.md.  First correct path: one sample per thread, the 17-dim state in
// registers, a general 4-stage RK4 (the drag makes v' depend on v, so the triangular short-cuts of
// rk4_step do not apply), the same objectives and the same fused softmax update as rollout_kernel.
#include <type_traits>
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
    ThrustDiff D = thrust_diff(T);                                       // the torques' thrust combinations (mppi_rate.cuh)
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
    const bool stored = (FUSED && OBJ != OBJ_CONTOUR_PAPER) ? keeps_du<STORE_DU>(A, b) : STORE_DU;
    float4* du_out = stored ? A.du + (size_t)b * N * P.K + k : nullptr;
    // the horizon loop, instantiated for the axisymmetric drag form (drag_x == drag_y) and the general one
    auto horizon = [&](auto axi) {
    for (int t = 0; t < N; ++t) {
        const float4 un = s_unom[t];
        const float4 u = sample_input<MATH>(P, A.rk, (uint32_t)k, (uint32_t)t, A.iter, (uint32_t)b, un, lo, hi);
        if (stored) du_out[(size_t)t * P.K] = make_float4(u.x - un.x, u.y - un.y, u.z - un.z, u.w - un.w);
        if (OBJ == OBJ_TRACK)      // eq.(8): the input term acts on the inputs = the rates [R-32]
            J += fmaf(P.R, u.x * u.x + u.y * u.y + u.z * u.z + u.w * u.w, track_state_term(P, s_trk + 4 * t, x));
        if (OBJ == OBJ_CONTOUR_PAPER) {            // fifth sampled input, stage cost, progress states [R-34]..[R-37]
            const float dv = sample_progress_accel<MATH>(P, A.rk, (uint32_t)k, (uint32_t)t, A.iter, (uint32_t)b,
                                                         s_vnom[t]);
            J += contour_paper_stage(P, s_trk, x, theta, v_theta, u, dv);
            theta = fmaf(P.hh2, dv, fmaf(P.dt, v_theta, theta));
            v_theta = fminf(fmaxf(fmaf(P.dt, dv, v_theta), 0.0f), P.v_theta_max);
        }
        rk4_rate_step<decltype(axi)::value>(P, x, T, D, u);
        J += rate_limit_cost(P, x);
        if (OBJ == OBJ_GATE) gc.template step<MATH>(P, s_trk, x);
        if (OBJ == OBJ_GATE_PAPER) gp.step(P, s_trk, s_front, x, t);
        if (OBJ == OBJ_CONTOUR) J += cc.step(P, s_trk, x);
    }
    };
    if (P.drag_x == P.drag_y) horizon(std::true_type{}); else horizon(std::false_type{});
    if (OBJ == OBJ_GATE) J += gc.finish<MATH>(P, s_trk, x);
    if (OBJ == OBJ_GATE_PAPER) J += gp.finish(P);
    if (OBJ == OBJ_TRACK) J += track_state_term(P, s_trk + 4 * N, x);
    J = sanitize_cost(J);
    A.cost[(size_t)b * P.K + k] = J;

    if (!FUSED) return;
    if (OBJ == OBJ_CONTOUR_PAPER)
        block_partial_and_combine<MATH>(P, A, b, blockIdx.x, J, lo, hi, s_unom, s_red, s_acc, s_pair, s_vnom, s_acc5);
    else
        block_partial_and_combine<MATH>(P, A, b, blockIdx.x, J, lo, hi, s_unom, s_red, s_acc, s_pair, nullptr, nullptr, stored);
}

// ---------------------------------------------------------------------------------------------
// packed throughput variant of the rate model: two samples per thread in fp32x2 registers
// (mppi_rate.cuh: fdyn_general2 / rk4_rate_step2).  grid = (K / (2 blockDim.x), B); thread j of the grid
// row owns samples 2j and 2j+1.  Objectives: gate, the paper's J_gate, tracking, the paper's contouring (eq.(9): theta,
// v_theta as packed states, the path looked up per half, the fifth input's column in the fused partial).
// ---------------------------------------------------------------------------------------------
template <int OBJ, int MATH, bool STORE_DU, bool FUSED>
__global__ void __launch_bounds__(128, 3) rollout_rate2_kernel(const DevParams P, const StepArgs A)
{
    extern __shared__ float4 smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int b = blockIdx.y;
    const int k0 = 2 * (blockIdx.x * blockDim.x + tid);
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
    const State x0 = load_state(xb);
    State2 x = splat_state(x0);
    float2 T[4] = { bc2(xb[13]), bc2(xb[14]), bc2(xb[15]), bc2(xb[16]) };
    ThrustDiff2 D = thrust_diff2(T[0], T[1], T[2], T[3]);
    float2 theta = bc2(0.0f), v_theta = bc2(0.0f);                       // OBJ_CONTOUR_PAPER: progress states [R-33]
    if (OBJ == OBJ_CONTOUR_PAPER) { theta = bc2(xb[17]); v_theta = bc2(xb[18]); }
    const float lo = -P.rate_max, hi = P.rate_max;

    float Ja = 0.0f, Jb = 0.0f;
    GateCost ga, gb;
    GatePaperCost pa, pb;
    const int* s_front = reinterpret_cast<const int*>(s_trk + 4 * P.G);  // OBJ_GATE_PAPER only
    if (OBJ == OBJ_GATE) { ga.init<MATH>(P, s_trk, start, x0); gb = ga; }
    if (OBJ == OBJ_GATE_PAPER) { pa.init(P, s_trk, start, x0); pb = pa; }
    const bool stored = (FUSED && OBJ != OBJ_CONTOUR_PAPER) ? keeps_du<STORE_DU>(A, b) : STORE_DU;
    float4* du_out = stored ? A.du + (size_t)b * N * P.K + k0 : nullptr;
    auto horizon = [&](auto axi) {         // as in rollout_rate_kernel: axisymmetric drag form / general form
    for (int t = 0; t < N; ++t) {
        const float4 un = s_unom[t];
        const float4 ua = sample_input<MATH>(P, A.rk, (uint32_t)k0, (uint32_t)t, A.iter, (uint32_t)b, un, lo, hi);
        const float4 ub = sample_input<MATH>(P, A.rk, (uint32_t)k0 + 1u, (uint32_t)t, A.iter, (uint32_t)b, un, lo, hi);
        if (stored) {
            du_out[(size_t)t * P.K] = make_float4(ua.x - un.x, ua.y - un.y, ua.z - un.z, ua.w - un.w);
            du_out[(size_t)t * P.K + 1] = make_float4(ub.x - un.x, ub.y - un.y, ub.z - un.z, ub.w - un.w);
        }
        if (OBJ == OBJ_TRACK) {
            Ja += fmaf(P.R, ua.x * ua.x + ua.y * ua.y + ua.z * ua.z + ua.w * ua.w, track_state_term(P, s_trk + 4 * t, lane_state<0>(x)));
            Jb += fmaf(P.R, ub.x * ub.x + ub.y * ub.y + ub.z * ub.z + ub.w * ub.w, track_state_term(P, s_trk + 4 * t, lane_state<1>(x)));
        }
        if (OBJ == OBJ_CONTOUR_PAPER) {            // fifth sampled input, stage cost, progress states [R-34]..[R-37]
            const float vn = s_vnom[t];
            const float dva = sample_progress_accel<MATH>(P, A.rk, (uint32_t)k0, (uint32_t)t, A.iter, (uint32_t)b, vn);
            const float dvb = sample_progress_accel<MATH>(P, A.rk, (uint32_t)k0 + 1u, (uint32_t)t, A.iter, (uint32_t)b, vn);
            Ja += contour_paper_stage(P, s_trk, lane_state<0>(x), theta.x, v_theta.x, ua, dva);
            Jb += contour_paper_stage(P, s_trk, lane_state<1>(x), theta.y, v_theta.y, ub, dvb);
            theta.x = fmaf(P.hh2, dva, fmaf(P.dt, v_theta.x, theta.x));
            theta.y = fmaf(P.hh2, dvb, fmaf(P.dt, v_theta.y, theta.y));
            v_theta.x = fminf(fmaxf(fmaf(P.dt, dva, v_theta.x), 0.0f), P.v_theta_max);
            v_theta.y = fminf(fmaxf(fmaf(P.dt, dvb, v_theta.y), 0.0f), P.v_theta_max);
        }
        rk4_rate_step2<decltype(axi)::value>(P, x, T, D, ua, ub);
        const State xa = lane_state<0>(x), xc = lane_state<1>(x);
        Ja += rate_limit_cost(P, xa);
        Jb += rate_limit_cost(P, xc);
        if (OBJ == OBJ_GATE) { ga.template step<MATH>(P, s_trk, xa); gb.template step<MATH>(P, s_trk, xc); }
        if (OBJ == OBJ_GATE_PAPER) { pa.step(P, s_trk, s_front, xa, t); pb.step(P, s_trk, s_front, xc, t); }
    }
    };
    if (P.drag_x == P.drag_y) horizon(std::true_type{}); else horizon(std::false_type{});
    if (OBJ == OBJ_GATE) { Ja += ga.finish<MATH>(P, s_trk, lane_state<0>(x)); Jb += gb.finish<MATH>(P, s_trk, lane_state<1>(x)); }
    if (OBJ == OBJ_GATE_PAPER) { Ja += pa.finish(P); Jb += pb.finish(P); }
    if (OBJ == OBJ_TRACK) {
        Ja += track_state_term(P, s_trk + 4 * N, lane_state<0>(x));
        Jb += track_state_term(P, s_trk + 4 * N, lane_state<1>(x));
    }
    Ja = sanitize_cost(Ja); Jb = sanitize_cost(Jb);
    *reinterpret_cast<float2*>(A.cost + (size_t)b * P.K + k0) = make_float2(Ja, Jb);

    if (!FUSED) return;

    // ---- block-local softmax partial over the block's 2 blockDim.x samples + last-block combine (mppi_rollout.cuh) ----
    const float Jv[2] = {Ja, Jb};
    if (OBJ == OBJ_CONTOUR_PAPER)
        block_partial_and_combine_n<MATH, 2>(P, A, b, blockIdx.x, (uint32_t)(2 * blockIdx.x * blockDim.x), Jv, lo, hi, false,
                                             s_unom, s_red, s_acc, s_pair, s_vnom, s_acc5);
    else
        block_partial_and_combine_n<MATH, 2>(P, A, b, blockIdx.x, (uint32_t)(2 * blockIdx.x * blockDim.x), Jv, lo, hi, stored,
                                             s_unom, s_red, s_acc, s_pair);
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

template <int OBJ, int MATH>
static RateFn pick_rate2p2(const LaunchCfg& c)
{
    if (c.fused) return c.store_du ? rollout_rate2_kernel<OBJ, MATH, true, true> : rollout_rate2_kernel<OBJ, MATH, false, true>;
    return rollout_rate2_kernel<OBJ, MATH, true, false>;
}
template <int OBJ>
static RateFn pick_rate2p1(const LaunchCfg& c)
{
    return c.fast_math ? pick_rate2p2<OBJ, 1>(c) : pick_rate2p2<OBJ, 0>(c);
}
static RateFn pick_rate_packed(const LaunchCfg& c)
{
    switch (c.objective) {
        case OBJ_GATE: return pick_rate2p1<OBJ_GATE>(c);
        case OBJ_GATE_PAPER: return pick_rate2p1<OBJ_GATE_PAPER>(c);
        case OBJ_CONTOUR_PAPER: return pick_rate2p1<OBJ_CONTOUR_PAPER>(c);
        default: return pick_rate2p1<OBJ_TRACK>(c);
    }
}

static RateFn pick_any(const LaunchCfg& c) { return c.pipe ? pick_pipe_rate(c) : c.packed ? pick_rate_packed(c) : pick_rate(c); }

const void* rate_kernel_ptr(const LaunchCfg& c) { return reinterpret_cast<const void*>(pick_any(c)); }

cudaError_t launch_rate(const DevParams& P, const StepArgs& A, const LaunchCfg& c, cudaStream_t s)
{
    pick_any(c)<<<dim3(P.blocks_per_ctrl, P.B), c.block_threads, c.smem_bytes, s>>>(P, A);
    return cudaGetLastError();
}

}  // namespace mppi
