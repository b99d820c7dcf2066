// mppi_pipe_rate.cuh -- the pipelined latency kernel for the paper's OWN input model (input_model = 1:
// thrust rates in, thrust states, rotor drag, soft body-rate limit; readings R-27..R-32 of DESIGN.md).
//
// Same idea as mppi_pipe.cuh -- one rollout cut into short dependent chains that run on different SM
// sub-partitions and are pipelined over the horizon steps through shared-memory rings -- but the drag
// term - R D R^T v of eq.(2) makes v' depend on v, so the translation is no longer a sum
// of thrust directions: it is split into a feed-forward part (the drag matrix M_i = R(q_i) D R(q_i)^T
// and the thrust acceleration a_i = c_i R(q_i) e_3 - g e_3 of every RK4 stage: two warps, alternate
// steps) and the short chain k_i = a_i - M_i v_i with the objective:
//
//   warps 4,5,6,8,9  draw the block's 32 x N clamped thrust RATES (eq.(3), [R-28]) into shared memory
//   warp 0 (W)   thrust states + body-rate chain: stage rates, collective accelerations -> ring W (16 floats)
//   warp 1 (Q)   attitude chain: the four stage quaternions (+ W's collective accelerations) -> ring Q (20 floats)
//   warps 3,7 (F) per stage M_i (6) and a_i (3), even / odd steps                          -> ring F (36 floats)
//   warp 2 (P)   velocity / position chain, position part of the objective
//
// Rings are handed over in chunks of kPipeChunk steps as in mppi_pipe.cuh.  The trajectory agrees with
// rk4_rate_step to rounding (M v instead of projecting v on the three body axes), not bit for bit.
// Block = 320 threads = 32 samples; grid = (K / 32, B).  Objectives: gate, the paper's J_gate, tracking, and
// the paper's own contouring (objective 4: the noise warps also draw the progress acceleration, W adds the
// input terms of eq.(9), P carries theta and v_theta and looks the path up; the fifth column of the
// update rides in the fused combine as in mppi_rate.cu).
#pragma once
#include "mppi_pipe.cuh"
#include "mppi_rate.cuh"

namespace mppi {

constexpr int kPipeRateThreads = 320;
// ring depths (chunks in flight) are launch parameters: (4, 3) when the grid is at most one block per SM
// (190 KB at N = 50), (2, 2) so that two blocks share an SM when the grid is up to twice the SM count
// (short horizons: the paper's Table I sizes, M = 8192, K = 20)

// float4 units of dynamic shared memory after the nominal + track + 16 float4 of reduction scratch
__host__ __device__ inline size_t pipe_rate_extra_f4(int N, int nb, bool progress, int d, int df)
{
    const int nchunks = (N + kPipeChunk - 1) / kPipeChunk;
    return (size_t)N * 33                                       // s_T   [N][33] thrust rates
           + (progress ? ((size_t)N * 33 + 3) / 4 : 0)          // s_dv  [N][32] progress accelerations, s_vnom [N]
           + (size_t)d * kPipeChunk * 4 * 32                    // ring W
           + (size_t)d * kPipeChunk * 5 * 32                    // ring Q
           + (size_t)df * kPipeChunk * 9 * 32                   // ring F
           + 32 + 8                                             // s_J [4][32], s_e [32]
           + (size_t)(3 * nb + 3) / 4                           // combine scratch
           + (size_t)(nchunks + 4 * d + 2 * df + 1) / 2;        // mbarriers (8 B each)
}

#define MPPI_G(QW, QX, QY, QZ, OX, OY, OZ, GW, GX, GY, GZ)                 \
    GW = fmaf(-(QZ), OZ, fmaf(-(QY), OY, -(QX) * (OX)));                   \
    GX = fmaf(-(QZ), OY, fmaf(QY, OZ, (QW) * (OX)));                       \
    GY = fmaf(-(QX), OZ, fmaf(QZ, OX, (QW) * (OY)));                       \
    GZ = fmaf(-(QY), OX, fmaf(QX, OY, (QW) * (OZ)));

// M = R D R^T (symmetric: xx xy xz yy yz zz) and a = c R e_3 - g e_3 for the stage quaternion q (not
// normalised at the inner stages: R(q) by the same polynomial as fdyn_general) -> 9 floats at f[0..8]
__device__ __forceinline__ void stage_force(const DevParams& P, const float4 q /* w x y z */, const float c, float* f)
{
    const float qw = q.x, qx = q.y, qy = q.z, qz = q.w;
    const float c0x = 1.0f - 2.0f * (qy * qy + qz * qz), c0y = 2.0f * (qx * qy + qw * qz), c0z = 2.0f * (qx * qz - qw * qy);
    const float c1x = 2.0f * (qx * qy - qw * qz), c1y = 1.0f - 2.0f * (qx * qx + qz * qz), c1z = 2.0f * (qy * qz + qw * qx);
    const float c2x = 2.0f * (qx * qz + qw * qy), c2y = 2.0f * (qy * qz - qw * qx), c2z = 1.0f - 2.0f * (qx * qx + qy * qy);
    const float s0x = P.drag_x * c0x, s0y = P.drag_x * c0y, s0z = P.drag_x * c0z;
    const float s1x = P.drag_y * c1x, s1y = P.drag_y * c1y, s1z = P.drag_y * c1z;
    const float s2x = P.drag_z * c2x, s2y = P.drag_z * c2y, s2z = P.drag_z * c2z;
    f[0] = fmaf(s2x, c2x, fmaf(s1x, c1x, s0x * c0x));
    f[1] = fmaf(s2x, c2y, fmaf(s1x, c1y, s0x * c0y));
    f[2] = fmaf(s2x, c2z, fmaf(s1x, c1z, s0x * c0z));
    f[3] = fmaf(s2y, c2y, fmaf(s1y, c1y, s0y * c0y));
    f[4] = fmaf(s2y, c2z, fmaf(s1y, c1z, s0y * c0z));
    f[5] = fmaf(s2z, c2z, fmaf(s1z, c1z, s0z * c0z));
    f[6] = c * c2x; f[7] = c * c2y; f[8] = fmaf(c, c2z, -P.g);
}

template <int OBJ, int MATH, bool STORE_DU, bool SHALLOW>
__global__ void __launch_bounds__(kPipeRateThreads, SHALLOW ? 2 : 1) rollout_pipe_rate_kernel(const DevParams P, const StepArgs A)
{
    extern __shared__ float4 smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int b = blockIdx.y, N = P.N;
    constexpr int RS = 33, C = kPipeChunk;
    constexpr int D = SHALLOW ? 2 : 4, DF = SHALLOW ? 2 : 3;      // = P.pipe_d, P.pipe_df (the host sizes the rings with those)
    const int kbase = blockIdx.x * 32;
    const int nchunks = (N + C - 1) / C;

    float4* s_unom = smem;
    float4* s_trk = smem + N;
    float* s_red = reinterpret_cast<float*>(s_trk + track_f4(P, OBJ));   // 64 floats
    float4* s_T = reinterpret_cast<float4*>(s_red + 64);                 // [N][RS] thrust rates
    float* s_dv = reinterpret_cast<float*>(s_T + (size_t)N * RS);        // OBJ_CONTOUR_PAPER: [N][32], then s_vnom [N]
    float* s_vnom = s_dv + (size_t)N * 32;
    float4* s_w = s_T + (size_t)N * RS + (OBJ == OBJ_CONTOUR_PAPER ? ((size_t)N * 33 + 3) / 4 : 0);   // [D][C][4][32]
    float4* s_q = s_w + D * C * 4 * 32;                                  // [D][C][5][32]
    float4* s_f = s_q + D * C * 5 * 32;                                  // [DF][C][9][32]
    float* s_J = reinterpret_cast<float*>(s_f + DF * C * 9 * 32);        // [4][32]
    float* s_e = s_J + 128;                                              // [32]
    float* s_pair = s_e + 32;                                            // 3 nb floats
    uint64_t* bar_T = reinterpret_cast<uint64_t*>(reinterpret_cast<float4*>(s_pair) + (3 * P.blocks_per_ctrl + 3) / 4);
    uint64_t* bar_wf = bar_T + nchunks;    // ring W full / empty, ring Q full / empty, ring F full / empty
    uint64_t* bar_we = bar_wf + D;
    uint64_t* bar_qf = bar_we + D;
    uint64_t* bar_qe = bar_qf + D;
    uint64_t* bar_ff = bar_qe + D;
    uint64_t* bar_fe = bar_ff + DF;

    const int start = A.start[b];
    stage_inputs<OBJ>(P, A, b, start, s_unom, s_trk);
    for (int i = tid; i < nchunks + 4 * D + 2 * DF; i += kPipeRateThreads) {
        uint32_t cnt = 32;
        if (i < nchunks) cnt = 32 * min(C, N - i * C);                       // every drawn (step, lane)
        else if (i >= nchunks + 3 * D && i < nchunks + 4 * D + DF) cnt = 64;    // Q empty, F full: both F warps
        mbar_init(bar_T + i, cnt);
    }
    if (OBJ == OBJ_CONTOUR_PAPER)
        for (int t = tid; t < N; t += kPipeRateThreads) s_vnom[t] = A.v_nom[(size_t)b * N + t];
    const float* xb = A.x0 + (OBJ == OBJ_CONTOUR_PAPER ? 19 : 17) * b;     // p, q, v, omega, T(4) [, theta, v_theta]
    const State x0 = load_state(xb);
    __syncthreads();

    const bool is_noise = warp == 4 || warp == 5 || warp == 6 || warp == 8 || warp == 9;
    if (is_noise) {
        // ---- noise producers: five warps, step t drawn by producer t % 5, one sample per lane (eq.(3)) ----
        const int w5 = warp < 7 ? warp - 4 : warp - 5;
        for (int t = w5; t < N; t += kPipeNoiseWarps) {
            const float4 un = s_unom[t];
            const float4 u = sample_input<MATH>(P, A.rk, (uint32_t)(kbase + lane), (uint32_t)t, A.iter, (uint32_t)b, un,
                                                -P.rate_max, P.rate_max);
            s_T[t * RS + lane] = u;
            if (OBJ == OBJ_CONTOUR_PAPER)       // the fifth sampled input [R-35]
                s_dv[t * 32 + lane] = sample_progress_accel<MATH>(P, A.rk, (uint32_t)(kbase + lane), (uint32_t)t, A.iter,
                                                                  (uint32_t)b, s_vnom[t]);
            mbar_arrive(bar_T + t / C);
            if (STORE_DU)
                A.du[((size_t)b * N + t) * P.K + kbase + lane] = make_float4(u.x - un.x, u.y - un.y, u.z - un.z, u.w - un.w);
        }
    } else if (warp == 0) {
        // ---- W: thrust states [R-27],[R-29] and body rates.  omega' = J^-1 (tau(T) - omega x J omega) ----
        float ox = x0.ox, oy = x0.oy, oz = x0.oz;
        float4 T = make_float4(xb[13], xb[14], xb[15], xb[16]);
        ThrustDiff TD = thrust_diff(T);            // the torques' thrust combinations, integrated beside T (mppi_rate.cuh)
        float acc = 0.0f, lim = 0.0f;
        for (int c = 0, s = 0, ph = 0; c < nchunks; ++c, ph ^= (s + 1 == D), s = (s + 1 == D) ? 0 : s + 1) {
            const int cnt = min(C, N - c * C);       // s = c % D, ph = (c / D) & 1, kept as running counters
            mbar_wait2(bar_T + c, 0, bar_we + s, ph ^ 1);
            for (int j = 0; j < cnt; ++j) {
                const int t = c * C + j;
                const float4 u = s_T[t * RS + lane];
                if (OBJ == OBJ_TRACK) {            // eq.(8): body-rate error at the pre-step state, R on the rates [R-32]
                    const float4 r2 = s_trk[4 * t + 2], r3 = s_trk[4 * t + 3];
                    const float wx = ox - r2.z, wy = oy - r2.w, wz = oz - r3.x;
                    acc = fmaf(P.Qw, wx * wx + wy * wy + wz * wz, acc);
                    acc = fmaf(P.R, u.x * u.x + u.y * u.y + u.z * u.z + u.w * u.w, acc);
                }
                if (OBJ == OBJ_CONTOUR_PAPER) {    // eq.(9): body-rate and input terms at the pre-step state [R-37]
                    const float dv = s_dv[t * 32 + lane];
                    acc = fmaf(P.w_omega, fmaf(oz, oz, fmaf(oy, oy, ox * ox)), acc);
                    acc = fmaf(P.r_dv, dv * dv, acc);
                    acc = fmaf(P.R, fmaf(u.w, u.w, fmaf(u.z, u.z, fmaf(u.y, u.y, u.x * u.x))), acc);
                }
                // torque accelerations and collective acceleration are linear in the thrusts: value at T and slope along u
                const ThrustDiff du = thrust_diff(u);
                const float ax = P.ltx * TD.x, bx = P.ltx * du.x;
                const float ay = P.lty * TD.y, by = P.lty * du.y;
                const float az = P.ltz * TD.z, bz = P.ltz * du.z;
                const float c0 = ((T.x + T.y) + (T.z + T.w)) * P.inv_mass, cu = ((u.x + u.y) + (u.z + u.w)) * P.inv_mass;
                const float amx = fmaf(P.h2, bx, ax), amy = fmaf(P.h2, by, ay), amz = fmaf(P.h2, bz, az);
                const float aex = fmaf(P.dt, bx, ax), aey = fmaf(P.dt, by, ay), aez = fmaf(P.dt, bz, az);
                float kx = fmaf(P.gyx, oy * oz, ax), ky = fmaf(P.gyy, oz * ox, ay), kz = fmaf(P.gyz, ox * oy, az);
                float nx = fmaf(P.h6, kx, ox), ny = fmaf(P.h6, ky, oy), nz = fmaf(P.h6, kz, oz);
                const float o2x = fmaf(P.h2, kx, ox), o2y = fmaf(P.h2, ky, oy), o2z = fmaf(P.h2, kz, oz);
                kx = fmaf(P.gyx, o2y * o2z, amx); ky = fmaf(P.gyy, o2z * o2x, amy); kz = fmaf(P.gyz, o2x * o2y, amz);
                nx = fmaf(P.h3, kx, nx); ny = fmaf(P.h3, ky, ny); nz = fmaf(P.h3, kz, nz);
                const float o3x = fmaf(P.h2, kx, ox), o3y = fmaf(P.h2, ky, oy), o3z = fmaf(P.h2, kz, oz);
                kx = fmaf(P.gyx, o3y * o3z, amx); ky = fmaf(P.gyy, o3z * o3x, amy); kz = fmaf(P.gyz, o3x * o3y, amz);
                nx = fmaf(P.h3, kx, nx); ny = fmaf(P.h3, ky, ny); nz = fmaf(P.h3, kz, nz);
                const float o4x = fmaf(P.dt, kx, ox), o4y = fmaf(P.dt, ky, oy), o4z = fmaf(P.dt, kz, oz);
                float4* w = s_w + (s * C + j) * 128 + lane;
                w[0] = make_float4(ox, oy, oz, o2x);
                w[32] = make_float4(o2y, o2z, o3x, o3y);
                w[64] = make_float4(o3z, o4x, o4y, o4z);
                w[96] = make_float4(c0, fmaf(P.h2, cu, c0), fmaf(P.dt, cu, c0), 0.0f);
                kx = fmaf(P.gyx, o4y * o4z, aex); ky = fmaf(P.gyy, o4z * o4x, aey); kz = fmaf(P.gyz, o4x * o4y, aez);
                ox = fmaf(P.h6, kx, nx); oy = fmaf(P.h6, ky, ny); oz = fmaf(P.h6, kz, nz);
                {   // thrust states: T + h u projected onto their range [R-29]; D follows its own rate unless the projection acted
                    const float4 Te = make_float4(fmaf(P.dt, u.x, T.x), fmaf(P.dt, u.y, T.y), fmaf(P.dt, u.z, T.z), fmaf(P.dt, u.w, T.w));
                    T.x = fminf(fmaxf(Te.x, P.T_min), P.T_max); T.y = fminf(fmaxf(Te.y, P.T_min), P.T_max);
                    T.z = fminf(fmaxf(Te.z, P.T_min), P.T_max); T.w = fminf(fmaxf(Te.w, P.T_min), P.T_max);
                    const bool moved = T.x != Te.x || T.y != Te.y || T.z != Te.z || T.w != Te.w;
                    const ThrustDiff Dc = thrust_diff(T);
                    TD.x = moved ? Dc.x : fmaf(P.dt, du.x, TD.x); TD.y = moved ? Dc.y : fmaf(P.dt, du.y, TD.y);
                    TD.z = moved ? Dc.z : fmaf(P.dt, du.z, TD.z);
                }
                {   // soft body-rate limit on the post-step rates [R-31]
                    const float ex = fmaxf(fabsf(ox) - P.omega_max, 0.0f), ey = fmaxf(fabsf(oy) - P.omega_max, 0.0f),
                                ez = fmaxf(fabsf(oz) - P.omega_max, 0.0f);
                    lim += P.w_limit * fmaf(ez, ez, fmaf(ey, ey, ex * ex));
                }
                if (OBJ == OBJ_GATE || OBJ == OBJ_GATE_PAPER) acc = fmaf(oz, oz, fmaf(oy, oy, fmaf(ox, ox, acc)));
            }
            mbar_arrive(bar_wf + s);
        }
        if (OBJ == OBJ_TRACK) {
            const float4 r2 = s_trk[4 * N + 2], r3 = s_trk[4 * N + 3];
            const float wx = ox - r2.z, wy = oy - r2.w, wz = oz - r3.x;
            acc = fmaf(P.Qw, wx * wx + wy * wy + wz * wz, acc);
        }
        s_J[lane] = acc;
        s_J[96 + lane] = lim;
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
        for (int c = 0, s = 0, ph = 0; c < nchunks; ++c, ph ^= (s + 1 == D), s = (s + 1 == D) ? 0 : s + 1) {
            const int cnt = min(C, N - c * C);
            mbar_wait2(bar_wf + s, ph, bar_qe + s, ph ^ 1);
            for (int j = 0; j < cnt; ++j) {
                if (OBJ == OBJ_TRACK) quat_term(s_trk + 4 * (c * C + j));
                const float4* w = s_w + (s * C + j) * 128 + lane;
                const float4 f0 = w[0], f1 = w[32], f2 = w[64], f3 = w[96];
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
                float4* o = s_q + (s * C + j) * 160 + lane;
                o[0] = make_float4(qw, qx, qy, qz);
                o[32] = make_float4(q2w, q2x, q2y, q2z);
                o[64] = make_float4(q3w, q3x, q3y, q3z);
                o[96] = make_float4(q4w, q4x, q4y, q4z);
                o[128] = f3;                                     // W's collective accelerations ride along
                MPPI_G(q4w, q4x, q4y, q4z, f2.y, f2.z, f2.w, gw, gx, gy, gz)
                nw = fmaf(P.h12, gw, nw); nx = fmaf(P.h12, gx, nx); ny = fmaf(P.h12, gy, ny); nz = fmaf(P.h12, gz, nz);
                const float inv = mufu_rsq(fmaf(nz, nz, fmaf(ny, ny, fmaf(nx, nx, nw * nw))));
                qw = nw * inv; qx = nx * inv; qy = ny * inv; qz = nz * inv;
            }
            mbar_arrive(bar_we + s);
            mbar_arrive(bar_qf + s);
        }
        if (OBJ == OBJ_TRACK) quat_term(s_trk + 4 * N);
        s_J[32 + lane] = acc;
    } else if (warp == 3 || warp == 7) {
        // ---- F: drag matrix and thrust acceleration of the four stages; warp 3 even steps, warp 7 odd ----
        const int par = warp == 3 ? 0 : 1;
        for (int c = 0, s = 0, ph = 0, sf = 0, phf = 0; c < nchunks;
             ++c, ph ^= (s + 1 == D), s = (s + 1 == D) ? 0 : s + 1, phf ^= (sf + 1 == DF), sf = (sf + 1 == DF) ? 0 : sf + 1) {
            const int cnt = min(C, N - c * C);
            mbar_wait2(bar_qf + s, ph, bar_fe + sf, phf ^ 1);
            for (int j = (c * C + par) & 1 ? 1 : 0; j < cnt; j += 2) {
                const float4* o = s_q + (s * C + j) * 160 + lane;
                const float4 cc = o[128];
                float f[36];
                stage_force(P, o[0], cc.x, f);
                stage_force(P, o[32], cc.y, f + 9);
                stage_force(P, o[64], cc.y, f + 18);
                stage_force(P, o[96], cc.z, f + 27);
                float4* g = s_f + (sf * C + j) * 288 + lane;
#pragma unroll
                for (int r = 0; r < 9; ++r) g[32 * r] = make_float4(f[4 * r], f[4 * r + 1], f[4 * r + 2], f[4 * r + 3]);
            }
            mbar_arrive(bar_qe + s);
            mbar_arrive(bar_ff + sf);
        }
    } else if (warp == 2) {
        // ---- P: velocity and position chain k_i = a_i - M_i v_i, position part of the objective ----
        State x = x0;
        x.ox = x.oy = x.oz = 0.0f;          // the body-rate terms are W's
        float J = 0.0f;
        GateCost gc;
        GatePaperCost gp;
        const int* s_front = reinterpret_cast<const int*>(s_trk + 4 * P.G);      // OBJ_GATE_PAPER only
        if (OBJ == OBJ_GATE) gc.init<MATH>(P, s_trk, start, x);
        if (OBJ == OBJ_GATE_PAPER) gp.init(P, s_trk, start, x);
        auto pv_term = [&](const float4* row) {
            const float4 a = row[0], r = row[1], r2 = row[2];
            const float ex = x.px - a.x, ey = x.py - a.y, ez = x.pz - a.z;
            const float ux = x.vx - r.w, uy = x.vy - r2.x, uz = x.vz - r2.y;
            J = fmaf(P.Qp, ex * ex + ey * ey + ez * ez, J);
            J = fmaf(P.Qv, ux * ux + uy * uy + uz * uz, J);
        };
        float theta = 0.0f, v_theta = 0.0f;                                  // OBJ_CONTOUR_PAPER: progress states [R-33]
        if (OBJ == OBJ_CONTOUR_PAPER) { theta = xb[17]; v_theta = xb[18]; }
        for (int c = 0, sf = 0, phf = 0; c < nchunks; ++c, phf ^= (sf + 1 == DF), sf = (sf + 1 == DF) ? 0 : sf + 1) {
            const int cnt = min(C, N - c * C);
            mbar_wait(bar_ff + sf, phf);
            for (int j = 0; j < cnt; ++j) {
                const int t = c * C + j;
                const float4* g = s_f + (sf * C + j) * 288 + lane;
                float f[36];
#pragma unroll
                for (int r = 0; r < 9; ++r) {
                    const float4 v4 = g[32 * r];
                    f[4 * r] = v4.x; f[4 * r + 1] = v4.y; f[4 * r + 2] = v4.z; f[4 * r + 3] = v4.w;
                }
                if (OBJ == OBJ_TRACK) pv_term(s_trk + 4 * t);
                if (OBJ == OBJ_CONTOUR_PAPER) {    // position part of eq.(9) at the pre-step state, progress states [R-34],[R-36]
                    float qx, qy, qz, tx, ty, tz;
                    path_eval(P, s_trk, theta, qx, qy, qz, tx, ty, tz);
                    const float ex = x.px - qx, ey = x.py - qy, ez = x.pz - qz;
                    const float e_l = fmaf(ez, tz, fmaf(ey, ty, ex * tx));
                    const float e_c2 = fmaxf(fmaf(ez, ez, fmaf(ey, ey, ex * ex)) - e_l * e_l, 0.0f);
                    J = fmaf(P.q_c, e_c2, fmaf(P.q_l * e_l, e_l, J));
                    J = fmaf(-P.mu, v_theta, J);
                    const float dv = s_dv[t * 32 + lane];
                    theta = fmaf(P.hh2, dv, fmaf(P.dt, v_theta, theta));
                    v_theta = fminf(fmaxf(fmaf(P.dt, dv, v_theta), 0.0f), P.v_theta_max);
                }
#define MPPI_K(F, VX, VY, VZ, KX, KY, KZ)                                                       \
    const float KX = fmaf(-(F)[2], VZ, fmaf(-(F)[1], VY, fmaf(-(F)[0], VX, (F)[6])));          \
    const float KY = fmaf(-(F)[4], VZ, fmaf(-(F)[3], VY, fmaf(-(F)[1], VX, (F)[7])));          \
    const float KZ = fmaf(-(F)[5], VZ, fmaf(-(F)[4], VY, fmaf(-(F)[2], VX, (F)[8])));
                MPPI_K(f, x.vx, x.vy, x.vz, k1x, k1y, k1z)
                const float v2x = fmaf(P.h2, k1x, x.vx), v2y = fmaf(P.h2, k1y, x.vy), v2z = fmaf(P.h2, k1z, x.vz);
                MPPI_K(f + 9, v2x, v2y, v2z, k2x, k2y, k2z)
                const float v3x = fmaf(P.h2, k2x, x.vx), v3y = fmaf(P.h2, k2y, x.vy), v3z = fmaf(P.h2, k2z, x.vz);
                MPPI_K(f + 18, v3x, v3y, v3z, k3x, k3y, k3z)
                const float v4x = fmaf(P.dt, k3x, x.vx), v4y = fmaf(P.dt, k3y, x.vy), v4z = fmaf(P.dt, k3z, x.vz);
                MPPI_K(f + 27, v4x, v4y, v4z, k4x, k4y, k4z)
#undef MPPI_K
                // p' = v: the stage velocities; v' = k
                x.px = fmaf(P.h6, (x.vx + v4x) + 2.0f * (v2x + v3x), x.px);
                x.py = fmaf(P.h6, (x.vy + v4y) + 2.0f * (v2y + v3y), x.py);
                x.pz = fmaf(P.h6, (x.vz + v4z) + 2.0f * (v2z + v3z), x.pz);
                x.vx = fmaf(P.h6, (k1x + k4x) + 2.0f * (k2x + k3x), x.vx);
                x.vy = fmaf(P.h6, (k1y + k4y) + 2.0f * (k2y + k3y), x.vy);
                x.vz = fmaf(P.h6, (k1z + k4z) + 2.0f * (k2z + k3z), x.vz);
                if (OBJ == OBJ_GATE) gc.step<MATH>(P, s_trk, x);
                if (OBJ == OBJ_GATE_PAPER) gp.step(P, s_trk, s_front, x, t);
            }
            mbar_arrive(bar_fe + sf);
        }
        if (OBJ == OBJ_GATE) J = gc.finish<MATH>(P, s_trk, x);
        if (OBJ == OBJ_GATE_PAPER) J = gp.finish(P);
        if (OBJ == OBJ_TRACK) pv_term(s_trk + 4 * N);
        s_J[64 + lane] = J;
    }
    __syncthreads();

    // ---- the parts of the cost meet; warp 0 owns the block's 32 samples from here on ----
    float m = 0.0f, Zb = 0.0f;
    if (warp == 0) {
        const float jw = s_J[lane], jq = s_J[32 + lane], jp = s_J[64 + lane], jl = s_J[96 + lane];
        float J;
        if (OBJ == OBJ_GATE || OBJ == OBJ_GATE_PAPER) J = fmaf(P.w_omega, jw, jp) + jl;
        else if (OBJ == OBJ_CONTOUR_PAPER) J = (jp + jw) + jl;
        else J = ((jp + jq) + jw) + jl;
        J = sanitize_cost(J);
        A.cost[(size_t)b * P.K + kbase + lane] = J;
        m = warp_min(J);
        const float e = exp_weight<MATH>((m - J) * P.inv_lambda);
        Zb = warp_sum(e);
        s_e[lane] = e;
    }
    __syncthreads();

    // ---- block partial S[t][i] = sum_l e_l (u_l[t][i] - u_nom[t][i]) from the rates in shared memory ----
    float* part = A.partials + ((size_t)b * P.blocks_per_ctrl + blockIdx.x) * P.part_stride;
    for (int j = tid; j < 4 * N; j += kPipeRateThreads) {
        const int t = j >> 2, i = j & 3;
        const float un = reinterpret_cast<const float*>(s_unom)[j];
        const float* row = reinterpret_cast<const float*>(s_T + t * RS) + i;
        float acc = 0.0f;
        for (int l = 0; l < 32; ++l) {
            const float el = s_e[l];                      // block-uniform
            if (el != 0.0f) acc = fmaf(el, row[4 * l] - un, acc);
        }
        part[j] = acc;
    }
    if (OBJ == OBJ_CONTOUR_PAPER)          // fifth column S5[t] = sum_l e_l (dv_l[t] - v_nom[t]), after the (m, Z) header
        for (int t = tid; t < N; t += kPipeRateThreads) {
            const float vn = s_vnom[t];
            float acc = 0.0f;
            for (int l = 0; l < 32; ++l) {
                const float el = s_e[l];
                if (el != 0.0f) acc = fmaf(el, s_dv[t * 32 + l] - vn, acc);
            }
            part[4 * N + 4 + t] = acc;
        }
    if (tid == 0) write_partial_header(P, A, b, blockIdx.x, m, Zb);
    publish_and_combine<MATH, (SHALLOW ? 2 : 4)>(P, A, b, P.blocks_per_ctrl, s_unom, s_red, s_pair, reinterpret_cast<float*>(s_T),
                              OBJ == OBJ_CONTOUR_PAPER ? s_vnom : nullptr);
}

#undef MPPI_G

}  // namespace mppi
