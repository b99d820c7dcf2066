// mppi_pipe.cuh -- the pipelined latency kernel: one rollout split over three warps.
//
// For a lone controller (configs[1]: K = 4096 -> 128 warps on 148 SMs) the iteration time is the
// dependent-issue chain of ONE warp: ~250 instructions per step with little ILP measured 490 cycles
// per step (profiles/README_r01.md).  eq.(2) is triangular --
//     omega' = f(omega, T)        q' = f(q, omega)        v' = f(q, T)        p' = v
// -- so the chain is cut into three shorter ones that run on three different SM sub-partitions and
// are pipelined over the horizon steps through shared-memory rings guarded by mbarriers:
//
//   warps 3..7  draw the block's 32 x N clamped thrusts (eq.(3)) into shared memory, step by step
//   warp 0 (W)  body-rate chain: the four RK4 stage rates of step t  -> ring W (12 floats / sample)
//   warp 1 (Q)  attitude chain:  the four RK4 stage quaternions      -> ring Q (16 floats / sample)
//   warp 2 (P)  translation: r(q_i) sums, p, v update, position part of the objective
//
// The rings are handed over in CHUNKS of kPipeChunk steps (one mbarrier wait + one arrive per chunk and
// side: a per-step handshake costs more than the arithmetic of a step -- measured), W runs ahead of Q
// and Q ahead of P by up to kPipeDepth chunks.  Every warp accumulates the terms
// of the objective that depend on its part of the state; they are added at the end.  The state
// trajectory is bit-identical to rk4_step (same operations in the same order per component).
// Block = 256 threads = 32 samples; grid = (K / 32, B).
#pragma once
#include "mppi_rollout.cuh"

namespace mppi {

constexpr int kPipeChunk = 5;      // steps per ring slot = steps per thrust mbarrier = noise warps
constexpr int kPipeDepth = 4;      // ring slots (chunks in flight between two stages of the pipeline)
constexpr int kPipeThreads = 256;
constexpr int kPipeNoiseWarps = kPipeChunk;

// ---- mbarrier helpers (CTA scope, shared memory) ------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@!p bra WAIT_%=;\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}

// two barriers at once: both phase checks are in flight together (a satisfied check costs ~100 cycles)
__device__ __forceinline__ void mbar_wait2(uint64_t* bar_a, uint32_t par_a, uint64_t* bar_b, uint32_t par_b)
{
    asm volatile(
        "{\n"
        ".reg .pred pa, pb;\n"
        "WAIT2_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 pa, [%0], %1;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 pb, [%2], %3;\n"
        "and.pred pa, pa, pb;\n"
        "@!pa bra WAIT2_%=;\n"
        "}\n" ::"r"(smem_u32(bar_a)), "r"(par_a), "r"(smem_u32(bar_b)), "r"(par_b) : "memory");
}

// float4 units of dynamic shared memory after the nominal + track + 16 float4 of reduction scratch
__host__ __device__ inline size_t pipe_extra_f4(int N, int nb)
{
    const int nchunks = (N + kPipeChunk - 1) / kPipeChunk;
    return (size_t)N * 33                                   // s_T   [N][33] thrusts
           + (size_t)kPipeDepth * kPipeChunk * 3 * 32       // ring W
           + (size_t)kPipeDepth * kPipeChunk * 4 * 32       // ring Q
           + 24 + 8                                         // s_J [3][32], s_e [32]
           + (size_t)(3 * nb + 3) / 4                       // combine scratch
           + (size_t)(nchunks + 4 * kPipeDepth + 1) / 2;    // mbarriers (8 B each)
}

// quaternion rate times two: G(q, w) = q (x) (0, w)    (the 1/2 is folded into the step constants)
#define MPPI_G(QW, QX, QY, QZ, OX, OY, OZ, GW, GX, GY, GZ)                 \
    GW = fmaf(-(QZ), OZ, fmaf(-(QY), OY, -(QX) * (OX)));                   \
    GX = fmaf(-(QZ), OY, fmaf(QY, OZ, (QW) * (OX)));                       \
    GY = fmaf(-(QX), OZ, fmaf(QZ, OX, (QW) * (OY)));                       \
    GZ = fmaf(-(QY), OX, fmaf(QX, OY, (QW) * (OZ)));

template <int OBJ, int MATH, bool STORE_DU>
__global__ void __launch_bounds__(kPipeThreads, 2) rollout_pipe_kernel(const DevParams P, const StepArgs A)
{
    extern __shared__ float4 smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int b = blockIdx.y, N = P.N;
    constexpr int RS = 33, D = kPipeDepth, C = kPipeChunk;
    const int kbase = blockIdx.x * 32;
    const int nchunks = (N + C - 1) / C;

    float4* s_unom = smem;
    float4* s_trk = smem + N;
    float* s_red = reinterpret_cast<float*>(s_trk + track_f4(P, OBJ));   // 64 floats
    float4* s_T = reinterpret_cast<float4*>(s_red + 64);                 // [N][RS]
    float4* s_w = s_T + (size_t)N * RS;                                  // [D][C][3][32]
    float4* s_q = s_w + D * C * 3 * 32;                                  // [D][C][4][32]
    float* s_J = reinterpret_cast<float*>(s_q + D * C * 4 * 32);         // [3][32]
    float* s_pair = s_J + 128;                                           // 3 nb floats (32 floats after s_J are spare)
    uint64_t* bar_T = reinterpret_cast<uint64_t*>(reinterpret_cast<float4*>(s_pair) + (3 * P.blocks_per_ctrl + 3) / 4);
    uint64_t* bar_wf = bar_T + nchunks;    // ring W full / empty, ring Q full / empty
    uint64_t* bar_we = bar_wf + D;
    uint64_t* bar_qf = bar_we + D;
    uint64_t* bar_qe = bar_qf + D;

    if (tid == 0) MPPI_STAMP(A, 0);
    // Programmatic dependent launch (mppi_optimize's chain): this kernel may have been started while the previous
    // kernel of the stream is still in its tail.  Everything that kernel neither writes nor reads comes first -- the
    // track, x0, the barriers and the state-independent half of the noise (Philox, radius, angle) -- then
    // griddepcontrol.wait, then the nominal (the previous kernel's output) and the rest as always.
    const bool pdl_wait = (A.pdl & 1) != 0;
    const int start = A.start[b];
    if (pdl_wait) stage_track<OBJ>(P, A, b, start, s_trk);
    else stage_inputs<OBJ>(P, A, b, start, s_unom, s_trk);
    for (int i = tid; i < nchunks + 4 * D; i += kPipeThreads)
        mbar_init(bar_T + i, i < nchunks ? 32 * min(C, N - i * C) : 32);
    const State x0 = load_state(A.x0 + 13 * b);
    if (pdl_wait) {
        if (warp >= 3)
            for (int t = warp - 3; t < N; t += kPipeNoiseWarps) {
                const uint4 r = philox4x32_10((uint32_t)(kbase + lane), (uint32_t)t, A.iter, (uint32_t)b, A.rk);
                float4 f;
                perturb_prepare<MATH>(r.x, r.y, P.bm_k, f.x, f.y);
                perturb_prepare<MATH>(r.z, r.w, P.bm_k, f.z, f.w);
                s_T[t * RS + lane] = f;
            }
        asm volatile("griddepcontrol.wait;" ::: "memory");
        stage_nominal(P, A, b, s_unom);
    }
    __syncthreads();
    const int i0 = OBJ == OBJ_CONTOUR ? contour_start_index(P, s_trk, start, x0, s_red) : 0;
    if (tid == 0) MPPI_STAMP(A, 1);

    if (warp >= 3) {
        // ---- noise producers: step t is drawn by warp 3 + t % 5, one sample per lane (eq.(3)) ----
        for (int t = warp - 3; t < N; t += kPipeNoiseWarps) {
            const float4 un = s_unom[t];
            float4 T;
            if (pdl_wait) {                        // second half of the pair drawn before the wait: the same operations
                const float4 f = s_T[t * RS + lane];
                perturb_finish<MATH>(f.x, f.y, P.sigma, un.x, un.y, T.x, T.y);
                perturb_finish<MATH>(f.z, f.w, P.sigma, un.z, un.w, T.z, T.w);
                T.x = fminf(fmaxf(T.x, P.T_min), P.T_max); T.y = fminf(fmaxf(T.y, P.T_min), P.T_max);
                T.z = fminf(fmaxf(T.z, P.T_min), P.T_max); T.w = fminf(fmaxf(T.w, P.T_min), P.T_max);
            } else {
                T = sample_thrust<MATH>(P, A.rk, (uint32_t)(kbase + lane), (uint32_t)t, A.iter, (uint32_t)b, un);
            }
            s_T[t * RS + lane] = T;
            mbar_arrive(bar_T + t / C);
            if (lane == 0 && t == 0) MPPI_STAMP(A, 2);
            if (lane == 0 && t == N - 1) MPPI_STAMP(A, 3);
            if (STORE_DU)
                A.du[((size_t)b * N + t) * P.K + kbase + lane] = make_float4(T.x - un.x, T.y - un.y, T.z - un.z, T.w - un.w);
        }
    } else if (warp == 0) {
        // ---- W: body rates.  omega' = J^-1 (tau - omega x J omega), PAPER.md:65-70 ----
        float ox = x0.ox, oy = x0.oy, oz = x0.oz;
        float acc = 0.0f;      // gate: sum |omega_{t+1}|^2; contour / track: this warp's cost terms
        for (int c = 0; c < nchunks; ++c) {
            const int s = c & (D - 1), cnt = min(C, N - c * C);
            // the chunk's thrusts are drawn; Q has drained this slot
            mbar_wait2(bar_T + c, 0, bar_we + s, ((c / D) & 1) ^ 1);
            for (int j = 0; j < cnt; ++j) {
                const int t = c * C + j;
                const float4 T = s_T[t * RS + lane];
                if (OBJ == OBJ_TRACK) {
                    const float4 r2 = s_trk[4 * t + 2], r3 = s_trk[4 * t + 3];
                    const float wx = ox - r2.z, wy = oy - r2.w, wz = oz - r3.x;
                    const float a0 = T.x - P.hover, a1 = T.y - P.hover, a2 = T.z - P.hover, a3 = T.w - P.hover;
                    acc = fmaf(P.Qw, wx * wx + wy * wy + wz * wz, acc);
                    acc = fmaf(P.R, a0 * a0 + a1 * a1 + a2 * a2 + a3 * a3, acc);
                }
                const float s01 = T.x + T.y, s23 = T.z + T.w;
                const float ax = P.ltx * (s01 - s23);
                const float d10 = T.y - T.x, d23 = T.z - T.w;
                const float ay = P.lty * (d10 + d23);
                const float az = P.ltz * (d23 - d10);
                float kx = fmaf(P.gyx, oy * oz, ax), ky = fmaf(P.gyy, oz * ox, ay), kz = fmaf(P.gyz, ox * oy, az);
                float nx = fmaf(P.h6, kx, ox), ny = fmaf(P.h6, ky, oy), nz = fmaf(P.h6, kz, oz);
                const float o2x = fmaf(P.h2, kx, ox), o2y = fmaf(P.h2, ky, oy), o2z = fmaf(P.h2, kz, oz);
                kx = fmaf(P.gyx, o2y * o2z, ax); ky = fmaf(P.gyy, o2z * o2x, ay); kz = fmaf(P.gyz, o2x * o2y, az);
                nx = fmaf(P.h3, kx, nx); ny = fmaf(P.h3, ky, ny); nz = fmaf(P.h3, kz, nz);
                const float o3x = fmaf(P.h2, kx, ox), o3y = fmaf(P.h2, ky, oy), o3z = fmaf(P.h2, kz, oz);
                kx = fmaf(P.gyx, o3y * o3z, ax); ky = fmaf(P.gyy, o3z * o3x, ay); kz = fmaf(P.gyz, o3x * o3y, az);
                nx = fmaf(P.h3, kx, nx); ny = fmaf(P.h3, ky, ny); nz = fmaf(P.h3, kz, nz);
                const float o4x = fmaf(P.dt, kx, ox), o4y = fmaf(P.dt, ky, oy), o4z = fmaf(P.dt, kz, oz);
                float4* w = s_w + (s * C + j) * 96 + lane;
                w[0] = make_float4(ox, oy, oz, o2x);
                w[32] = make_float4(o2y, o2z, o3x, o3y);
                w[64] = make_float4(o3z, o4x, o4y, o4z);
                kx = fmaf(P.gyx, o4y * o4z, ax); ky = fmaf(P.gyy, o4z * o4x, ay); kz = fmaf(P.gyz, o4x * o4y, az);
                ox = fmaf(P.h6, kx, nx); oy = fmaf(P.h6, ky, ny); oz = fmaf(P.h6, kz, nz);
                if (OBJ == OBJ_GATE || OBJ == OBJ_GATE_PAPER) acc = fmaf(oz, oz, fmaf(oy, oy, fmaf(ox, ox, acc)));
                if (OBJ == OBJ_CONTOUR) acc = fmaf(P.w_omega, ox * ox + oy * oy + oz * oz, acc);
            }
            mbar_arrive(bar_wf + s);
        }
        if (OBJ == OBJ_TRACK) {
            const float4 r2 = s_trk[4 * N + 2], r3 = s_trk[4 * N + 3];
            const float wx = ox - r2.z, wy = oy - r2.w, wz = oz - r3.x;
            acc = fmaf(P.Qw, wx * wx + wy * wy + wz * wz, acc);
        }
        s_J[lane] = acc;
        // the body-rate chain of this block is through: a dependent launch (the next iteration of mppi_optimize's chain)
        // may start on the SMs.  Measured per iteration of the 10-iteration chain: trigger here 14.0 us, after all
        // rollouts 14.8 us, at kernel start 15.7 us (its noise warps then compete with this kernel's chains); plain
        // launches 16.1 us, one graph launch 14.3 us.
        if (A.pdl & 2) asm volatile("griddepcontrol.launch_dependents;");
        if (lane == 0) MPPI_STAMP(A, 4);
    } else if (warp == 1) {
        // ---- Q: attitude.  q' = 1/2 q (x) (0, omega), renormalised once per step [R-5] ----
        float qw = x0.qw, qx = x0.qx, qy = x0.qy, qz = x0.qz;
        float acc = 0.0f;
        auto quat_term = [&](const float4* row) {
            const float4 a = row[0], r = row[1];
            const float dot = qw * a.w + qx * r.x + qy * r.y + qz * r.z;
            const float sg = dot < 0.0f ? -1.0f : 1.0f;
            const float e0 = fmaf(-sg, a.w, qw), e1 = fmaf(-sg, r.x, qx), e2 = fmaf(-sg, r.y, qy), e3 = fmaf(-sg, r.z, qz);
            acc = fmaf(P.Qq, e0 * e0 + e1 * e1 + e2 * e2 + e3 * e3, acc);
        };
        for (int c = 0; c < nchunks; ++c) {
            const int s = c & (D - 1), cnt = min(C, N - c * C);
            // W has filled this slot; P has drained the slot written below
            mbar_wait2(bar_wf + s, (c / D) & 1, bar_qe + s, ((c / D) & 1) ^ 1);
            for (int j = 0; j < cnt; ++j) {
                if (OBJ == OBJ_TRACK) quat_term(s_trk + 4 * (c * C + j));
                const float4* w = s_w + (s * C + j) * 96 + lane;
                const float4 f0 = w[0], f1 = w[32], f2 = w[64];
                float gw, gx, gy, gz;
                MPPI_G(qw, qx, qy, qz, f0.x, f0.y, f0.z, gw, gx, gy, gz)
                float nw = fmaf(P.h12, gw, qw), nx = fmaf(P.h12, gx, qx), ny = fmaf(P.h12, gy, qy), nz = fmaf(P.h12, gz, qz);
                const float q2w = fmaf(P.h4, gw, qw), q2x = fmaf(P.h4, gx, qx), q2y = fmaf(P.h4, gy, qy), q2z = fmaf(P.h4, gz, qz);
                MPPI_G(q2w, q2x, q2y, q2z, f0.w, f1.x, f1.y, gw, gx, gy, gz)
                nw = fmaf(P.h6, gw, nw); nx = fmaf(P.h6, gx, nx); ny = fmaf(P.h6, gy, ny); nz = fmaf(P.h6, gz, nz);
                const float q3w = fmaf(P.h4, gw, qw), q3x = fmaf(P.h4, gx, qx), q3y = fmaf(P.h4, gy, qy), q3z = fmaf(P.h4, gz, qz);
                MPPI_G(q3w, q3x, q3y, q3z, f1.z, f1.w, f2.x, gw, gx, gy, gz)
                nw = fmaf(P.h6, gw, nw); nx = fmaf(P.h6, gx, nx); ny = fmaf(P.h6, gy, ny); nz = fmaf(P.h6, gz, nz);
                const float q4w = fmaf(P.h2, gw, qw), q4x = fmaf(P.h2, gx, qx), q4y = fmaf(P.h2, gy, qy), q4z = fmaf(P.h2, gz, qz);
                float4* o = s_q + (s * C + j) * 128 + lane;
                o[0] = make_float4(qw, qx, qy, qz);
                o[32] = make_float4(q2w, q2x, q2y, q2z);
                o[64] = make_float4(q3w, q3x, q3y, q3z);
                o[96] = make_float4(q4w, q4x, q4y, q4z);
                MPPI_G(q4w, q4x, q4y, q4z, f2.y, f2.z, f2.w, gw, gx, gy, gz)
                nw = fmaf(P.h12, gw, nw); nx = fmaf(P.h12, gx, nx); ny = fmaf(P.h12, gy, ny); nz = fmaf(P.h12, gz, nz);
                // |n|^2 is within rounding of 1: the plain MUFU.RSQ (no denormal fix-up) returns rsqrtf's value
                const float inv = mufu_rsq(fmaf(nz, nz, fmaf(ny, ny, fmaf(nx, nx, nw * nw))));
                qw = nw * inv; qx = nx * inv; qy = ny * inv; qz = nz * inv;
            }
            mbar_arrive(bar_we + s);
            mbar_arrive(bar_qf + s);
        }
        if (OBJ == OBJ_TRACK) quat_term(s_trk + 4 * N);
        s_J[32 + lane] = acc;
        if (lane == 0) MPPI_STAMP(A, 5);
    } else {
        // ---- P: translation and the position part of the objective ----
        State x = x0;
        x.ox = x.oy = x.oz = 0.0f;          // the body-rate terms are W's
        float J = 0.0f;
        GateCost gc;
        GatePaperCost gp;
        ContourCost cc;
        const int* s_front = reinterpret_cast<const int*>(s_trk + 4 * P.G);      // OBJ_GATE_PAPER only
        if (OBJ == OBJ_GATE) gc.init<MATH>(P, s_trk, start, x);
        if (OBJ == OBJ_GATE_PAPER) gp.init(P, s_trk, start, x);
        if (OBJ == OBJ_CONTOUR) cc.init(P, s_trk, i0, x);
        auto pv_term = [&](const float4* row) {
            const float4 a = row[0], r = row[1], r2 = row[2];
            const float ex = x.px - a.x, ey = x.py - a.y, ez = x.pz - a.z;
            const float ux = x.vx - r.w, uy = x.vy - r2.x, uz = x.vz - r2.y;
            J = fmaf(P.Qp, ex * ex + ey * ey + ez * ez, J);
            J = fmaf(P.Qv, ux * ux + uy * uy + uz * uz, J);
        };
        for (int c = 0; c < nchunks; ++c) {
            const int s = c & (D - 1), cnt = min(C, N - c * C);
            mbar_wait(bar_qf + s, (c / D) & 1);                // Q has filled this slot (its thrusts are older)
            for (int j = 0; j < cnt; ++j) {
                const int t = c * C + j;
                const float4 T = s_T[t * RS + lane];
                const float4* o = s_q + (s * C + j) * 128 + lane;
                const float4 q1 = o[0], q2 = o[32], q3 = o[64], q4 = o[96];
                if (OBJ == OBJ_TRACK) pv_term(s_trk + 4 * t);
                const float cm = ((T.x + T.y) + (T.z + T.w)) * P.inv_mass;
                const float cz0 = cm - P.g, kp = cm * P.hh3, kv = cm * P.h3;
#define MPPI_R(Q, RX, RY, RZ)                                                              \
    const float RX = fmaf(Q.x, Q.z, Q.y * Q.w), RY = fmaf(-Q.x, Q.y, Q.z * Q.w), RZ = fmaf(Q.z, Q.z, Q.y * Q.y);
                MPPI_R(q1, r1x, r1y, r1z) MPPI_R(q2, r2x, r2y, r2z) MPPI_R(q3, r3x, r3y, r3z) MPPI_R(q4, r4x, r4y, r4z)
#undef MPPI_R
                const float mx = r2x + r3x, my = r2y + r3y, mz = r2z + r3z;
                const float Ax = r1x + mx, Ay = r1y + my, Az = r1z + mz;
                x.px = fmaf(kp, Ax, fmaf(P.dt, x.vx, x.px));
                x.py = fmaf(kp, Ay, fmaf(P.dt, x.vy, x.py));
                x.pz = fmaf(-kp, Az, fmaf(P.hh2, cz0, fmaf(P.dt, x.vz, x.pz)));
                x.vx = fmaf(kv, (Ax + mx) + r4x, x.vx);
                x.vy = fmaf(kv, (Ay + my) + r4y, x.vy);
                x.vz = fmaf(-kv, (Az + mz) + r4z, fmaf(P.dt, cz0, x.vz));
                if (OBJ == OBJ_GATE) gc.step<MATH>(P, s_trk, x);
                if (OBJ == OBJ_GATE_PAPER) gp.step(P, s_trk, s_front, x, t);
                if (OBJ == OBJ_CONTOUR) J += cc.step(P, s_trk, x);
            }
            mbar_arrive(bar_qe + s);
        }
        if (OBJ == OBJ_GATE) J = gc.finish<MATH>(P, s_trk, x);
        if (OBJ == OBJ_GATE_PAPER) J = gp.finish(P);
        if (OBJ == OBJ_TRACK) pv_term(s_trk + 4 * N);
        s_J[64 + lane] = J;
        if (lane == 0) MPPI_STAMP(A, 6);
    }
    __syncthreads();

    // ---- the three parts of the cost meet.  Every warp forms the 32 costs, their minimum and the weights e_l on its
    // own (three shared-memory reads and two shuffle reductions, the same values in every warp): no second barrier
    // and no round trip through shared memory before the partial ----
    const float jw = s_J[lane], jq = s_J[32 + lane], jp = s_J[64 + lane];
    float J;
    if (OBJ == OBJ_GATE || OBJ == OBJ_GATE_PAPER) J = fmaf(P.w_omega, jw, jp);   // = finish() with W's sum |omega|^2
    else if (OBJ == OBJ_TRACK) J = (jp + jq) + jw;
    else J = jp + jw;
    J = sanitize_cost(J);
    if (warp == 0) A.cost[(size_t)b * P.K + kbase + lane] = J;
    const float m = warp_min(J);
    const float e = exp_weight<MATH>((m - J) * P.inv_lambda);
    const float Zb = warp_sum(e);
    const unsigned contrib = __ballot_sync(kFull, e != 0.0f);

    // ---- block partial S[t][i] = sum_l e_l (T_l[t][i] - u_nom[t][i]) from the thrusts in shared memory: thread j
    // owns column j; only the samples with a non-zero weight are visited, in ascending order (e_l by shuffle) ----
    float* part = A.partials + ((size_t)b * P.blocks_per_ctrl + blockIdx.x) * P.part_stride;
    for (int j0 = warp * 32; j0 < 4 * N; j0 += kPipeThreads) {
        const int j = j0 + lane;
        const bool live = j < 4 * N;
        const int t = j >> 2, i = j & 3;
        const float un = live ? reinterpret_cast<const float*>(s_unom)[j] : 0.0f;
        const float* row = reinterpret_cast<const float*>(s_T + (live ? t : 0) * RS) + i;
        float acc = 0.0f;
        unsigned mm = contrib;
        while (mm) {
            const int l = __ffs(mm) - 1;
            mm &= mm - 1;
            acc = fmaf(__shfl_sync(kFull, e, l), row[4 * l] - un, acc);
        }
        if (live) part[j] = acc;
    }
    if (tid == 0) write_partial_header(P, A, b, blockIdx.x, m, Zb);
    if (tid == 0) MPPI_STAMP(A, 7);
    publish_and_combine<MATH, 4>(P, A, b, P.blocks_per_ctrl, s_unom, s_red, s_pair, reinterpret_cast<float*>(s_T));
    if (tid == 0) MPPI_STAMP(A, 12);
}

#undef MPPI_G

}  // namespace mppi
