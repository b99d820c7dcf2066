// mppi_rate.cu -- the rollout under the paper's OWN input model: the control input is
// the thrust RATE u = dT/dt and the four rotor thrusts are states ("Following the approach
// in [4] ..."), with the rate and thrust ranges of Table I, the rotor-drag term
// - R D R^T v of eq.(2) and a soft body-rate limit ("external cost").
// Readings R-27..R-32 of DESIGN.md.  First correct path: one sample per thread, the 17-dim state in
// registers, a general 4-stage RK4 (the drag makes v' depend on v, so the triangular short-cuts of
// rk4_step do not apply), the same objectives and the same fused softmax update as rollout_kernel.
#include "mppi_internal.h"
#include "mppi_rollout.cuh"

namespace mppi {

struct Deriv { float qw, qx, qy, qz, vx, vy, vz, ox, oy, oz; };     // p' = v needs no slot

// f_dyn of eq.(2) for the attitude, velocity and body-rate parts at stage state (q, v, o) with rotor
// thrusts T.  q' carries its 1/2 here (general form).
__device__ __forceinline__ Deriv fdyn_general(const DevParams& P, const float qw, const float qx, const float qy,
                                              const float qz, const float vx, const float vy, const float vz,
                                              const float ox, const float oy, const float oz, const float4 T)
{
    Deriv d;
    d.qw = 0.5f * fmaf(-qz, oz, fmaf(-qy, oy, -qx * ox));
    d.qx = 0.5f * fmaf(-qz, oy, fmaf(qy, oz, qw * ox));
    d.qy = 0.5f * fmaf(-qx, oz, fmaf(qz, ox, qw * oy));
    d.qz = 0.5f * fmaf(-qy, ox, fmaf(qx, oy, qw * oz));
    const float s01 = T.x + T.y, s23 = T.z + T.w;
    d.ox = fmaf(P.gyx, oy * oz, P.ltx * (s01 - s23));                  // PAPER.md:70, J^-1 folded in
    d.oy = fmaf(P.gyy, oz * ox, P.lty * ((T.y + T.z) - (T.x + T.w)));
    d.oz = fmaf(P.gyz, ox * oy, P.ltz * ((T.x + T.z) - (T.y + T.w)));
    // columns of R(q): the body axes in the world frame
    const float c0x = 1.0f - 2.0f * (qy * qy + qz * qz), c0y = 2.0f * (qx * qy + qw * qz), c0z = 2.0f * (qx * qz - qw * qy);
    const float c1x = 2.0f * (qx * qy - qw * qz), c1y = 1.0f - 2.0f * (qx * qx + qz * qz), c1z = 2.0f * (qy * qz + qw * qx);
    const float c2x = 2.0f * (qx * qz + qw * qy), c2y = 2.0f * (qy * qz - qw * qx), c2z = 1.0f - 2.0f * (qx * qx + qy * qy);
    const float c = (s01 + s23) * P.inv_mass;
    // - R D R^T v: project v on each body axis, scale by that axis' coefficient [R-30]
    const float b0 = P.drag_x * fmaf(c0z, vz, fmaf(c0y, vy, c0x * vx));
    const float b1 = P.drag_y * fmaf(c1z, vz, fmaf(c1y, vy, c1x * vx));
    const float b2 = P.drag_z * fmaf(c2z, vz, fmaf(c2y, vy, c2x * vx));
    d.vx = fmaf(c, c2x, -fmaf(c2x, b2, fmaf(c1x, b1, c0x * b0)));
    d.vy = fmaf(c, c2y, -fmaf(c2y, b2, fmaf(c1y, b1, c0y * b0)));
    d.vz = fmaf(c, c2z, -fmaf(c2z, b2, fmaf(c1z, b1, c0z * b0))) - P.g;
    return d;
}

// x <- RK4 on the 17-vector [p, q, v, omega, T] with T' = u held over the step; q renormalised; the
// thrust states projected onto [T_min, T_max] afterwards [R-27],[R-29].
__device__ __forceinline__ void rk4_rate_step(const DevParams& P, State& x, float4& T, const float4 u)
{
    const float h = P.dt, hh = P.h2;
    const float4 Tm = make_float4(fmaf(hh, u.x, T.x), fmaf(hh, u.y, T.y), fmaf(hh, u.z, T.z), fmaf(hh, u.w, T.w));
    const float4 Te = make_float4(fmaf(h, u.x, T.x), fmaf(h, u.y, T.y), fmaf(h, u.z, T.z), fmaf(h, u.w, T.w));
    // stage 1
    Deriv k = fdyn_general(P, x.qw, x.qx, x.qy, x.qz, x.vx, x.vy, x.vz, x.ox, x.oy, x.oz, T);
    float apx = x.vx, apy = x.vy, apz = x.vz;                         // sums of p' = v over the stages
    Deriv a = k;
    float vx = fmaf(hh, k.vx, x.vx), vy = fmaf(hh, k.vy, x.vy), vz = fmaf(hh, k.vz, x.vz);
    float qw = fmaf(hh, k.qw, x.qw), qx = fmaf(hh, k.qx, x.qx), qy = fmaf(hh, k.qy, x.qy), qz = fmaf(hh, k.qz, x.qz);
    float ox = fmaf(hh, k.ox, x.ox), oy = fmaf(hh, k.oy, x.oy), oz = fmaf(hh, k.oz, x.oz);
#define MPPI_ACC(W)                                                                                    \
    a.qw = fmaf(W, k.qw, a.qw); a.qx = fmaf(W, k.qx, a.qx); a.qy = fmaf(W, k.qy, a.qy); a.qz = fmaf(W, k.qz, a.qz); \
    a.vx = fmaf(W, k.vx, a.vx); a.vy = fmaf(W, k.vy, a.vy); a.vz = fmaf(W, k.vz, a.vz);               \
    a.ox = fmaf(W, k.ox, a.ox); a.oy = fmaf(W, k.oy, a.oy); a.oz = fmaf(W, k.oz, a.oz);
    // stage 2 (state x + h/2 k1, thrusts T + h/2 u)
    apx = fmaf(2.0f, vx, apx); apy = fmaf(2.0f, vy, apy); apz = fmaf(2.0f, vz, apz);
    k = fdyn_general(P, qw, qx, qy, qz, vx, vy, vz, ox, oy, oz, Tm);
    MPPI_ACC(2.0f)
    vx = fmaf(hh, k.vx, x.vx); vy = fmaf(hh, k.vy, x.vy); vz = fmaf(hh, k.vz, x.vz);
    qw = fmaf(hh, k.qw, x.qw); qx = fmaf(hh, k.qx, x.qx); qy = fmaf(hh, k.qy, x.qy); qz = fmaf(hh, k.qz, x.qz);
    ox = fmaf(hh, k.ox, x.ox); oy = fmaf(hh, k.oy, x.oy); oz = fmaf(hh, k.oz, x.oz);
    // stage 3
    apx = fmaf(2.0f, vx, apx); apy = fmaf(2.0f, vy, apy); apz = fmaf(2.0f, vz, apz);
    k = fdyn_general(P, qw, qx, qy, qz, vx, vy, vz, ox, oy, oz, Tm);
    MPPI_ACC(2.0f)
    vx = fmaf(h, k.vx, x.vx); vy = fmaf(h, k.vy, x.vy); vz = fmaf(h, k.vz, x.vz);
    qw = fmaf(h, k.qw, x.qw); qx = fmaf(h, k.qx, x.qx); qy = fmaf(h, k.qy, x.qy); qz = fmaf(h, k.qz, x.qz);
    ox = fmaf(h, k.ox, x.ox); oy = fmaf(h, k.oy, x.oy); oz = fmaf(h, k.oz, x.oz);
    // stage 4 (state x + h k3, thrusts T + h u)
    apx += vx; apy += vy; apz += vz;
    k = fdyn_general(P, qw, qx, qy, qz, vx, vy, vz, ox, oy, oz, Te);
    MPPI_ACC(1.0f)
#undef MPPI_ACC
    const float h6 = P.h6;
    x.px = fmaf(h6, apx, x.px); x.py = fmaf(h6, apy, x.py); x.pz = fmaf(h6, apz, x.pz);
    x.vx = fmaf(h6, a.vx, x.vx); x.vy = fmaf(h6, a.vy, x.vy); x.vz = fmaf(h6, a.vz, x.vz);
    x.ox = fmaf(h6, a.ox, x.ox); x.oy = fmaf(h6, a.oy, x.oy); x.oz = fmaf(h6, a.oz, x.oz);
    const float nw = fmaf(h6, a.qw, x.qw), nx = fmaf(h6, a.qx, x.qx), ny = fmaf(h6, a.qy, x.qy), nz = fmaf(h6, a.qz, x.qz);
    const float inv = rsqrtf(fmaf(nz, nz, fmaf(ny, ny, fmaf(nx, nx, nw * nw))));
    x.qw = nw * inv; x.qx = nx * inv; x.qy = ny * inv; x.qz = nz * inv;
    T.x = fminf(fmaxf(Te.x, P.T_min), P.T_max); T.y = fminf(fmaxf(Te.y, P.T_min), P.T_max);
    T.z = fminf(fmaxf(Te.z, P.T_min), P.T_max); T.w = fminf(fmaxf(Te.w, P.T_min), P.T_max);
}

// soft body-rate limit [R-31]
__device__ __forceinline__ float rate_limit_cost(const DevParams& P, const State& x)
{
    const float ex = fmaxf(fabsf(x.ox) - P.omega_max, 0.0f), ey = fmaxf(fabsf(x.oy) - P.omega_max, 0.0f),
                ez = fmaxf(fabsf(x.oz) - P.omega_max, 0.0f);
    return P.w_limit * fmaf(ez, ez, fmaf(ey, ey, ex * ex));
}

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

    const int start = A.start[b];
    stage_inputs<OBJ>(P, A, b, start, s_unom, s_trk);
    __syncthreads();

    const float* xb = A.x0 + 17 * b;                                     // p, q, v, omega, T(4)
    State x = load_state(xb);
    float4 T = make_float4(xb[13], xb[14], xb[15], xb[16]);
    const int i0 = OBJ == OBJ_CONTOUR ? contour_start_index(P, s_trk, start, x, s_red) : 0;
    const float lo = -P.rate_max, hi = P.rate_max;                       // [R-28]

    float J = 0.0f;
    GateCost gc;
    GatePaperCost gp;
    ContourCost cc;
    const int* s_front = reinterpret_cast<const int*>(s_trk + 4 * P.G);  // OBJ_GATE_PAPER only
    if (OBJ == OBJ_GATE) gc.init<MATH>(P, s_trk, start, x);
    if (OBJ == OBJ_GATE_PAPER) gp.init(P, s_trk, start, x);
    if (OBJ == OBJ_CONTOUR) cc.init(s_trk, i0, x);
    float4* du_out = STORE_DU ? A.du + (size_t)b * N * P.K + k : nullptr;
    for (int t = 0; t < N; ++t) {
        const float4 un = s_unom[t];
        const float4 u = sample_input<MATH>(P, A.rk, (uint32_t)k, (uint32_t)t, A.iter, (uint32_t)b, un, lo, hi);
        if (STORE_DU) du_out[(size_t)t * P.K] = make_float4(u.x - un.x, u.y - un.y, u.z - un.z, u.w - un.w);
        if (OBJ == OBJ_TRACK)      // eq.(8): the input term acts on the inputs = the rates [R-32]
            J += fmaf(P.R, u.x * u.x + u.y * u.y + u.z * u.z + u.w * u.w, track_state_term(P, s_trk + 4 * t, x));
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
        default: return pick_rate1<OBJ_CONTOUR>(c);
    }
}

const void* rate_kernel_ptr(const LaunchCfg& c) { return reinterpret_cast<const void*>(pick_rate(c)); }

cudaError_t launch_rate(const DevParams& P, const StepArgs& A, const LaunchCfg& c, cudaStream_t s)
{
    pick_rate(c)<<<dim3(P.blocks_per_ctrl, P.B), c.block_threads, c.smem_bytes, s>>>(P, A);
    return cudaGetLastError();
}

}  // namespace mppi
