// mppi_rate.cuh -- device functions of the paper's own input model:
// general f_dyn with rotor drag, RK4 on the 17-vector [p, q, v, omega, T], soft body-rate limit.
// Used by the rollout kernel (mppi_rate.cu) and by the plant / nominal-rollout kernels (mppi_kernels.cu).
#pragma once
#include "mppi_device.cuh"

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

// ---- the paper's own contouring formulation, eq.(9) PAPER.md:149-161 ----------------
// P(theta) and the unit tangent at theta from the path in shared memory (points (P_i, s_i), then tangents) [R-36]:
// theta wrapped into [0, L) on a closed path (clamped on an open one); the segment is found from the
// uniform-spacing guess theta P / L and corrected by stepping (the arc lengths are cumulative chord
// lengths, only nearly uniform); linear interpolation of the points, normalised linear interpolation
// of the vertex tangents.
__device__ __forceinline__ void path_eval(const DevParams& P, const float4* s_path, const float theta,
                                          float& px, float& py, float& pz, float& tx, float& ty, float& tz)
{
    const int n = P.P;
    float th = theta;
    if (P.closed) { th = fmaf(-P.path_L, floorf(th * P.inv_path_L), th); if (th >= P.path_L) th = 0.0f; if (th < 0.0f) th = 0.0f; }
    else th = fminf(fmaxf(th, 0.0f), s_path[n - 1].w);
    const int last = P.closed ? n - 1 : n - 2;
    int i = min(max((int)(th * P.inv_path_L * (float)n), 0), last);
    while (i > 0 && s_path[i].w > th) --i;
    while (i < last && s_path[i + 1].w <= th) ++i;
    const int j = (i + 1 == n) ? 0 : i + 1;
    const float4 a = s_path[i], b = s_path[j], ta = s_path[n + i], tb = s_path[n + j];
    const float s1 = (i + 1 < n) ? b.w : P.path_L;
    const float lam = fminf((th - a.w) / (s1 - a.w), 1.0f), mu = 1.0f - lam;
    px = fmaf(lam, b.x, mu * a.x); py = fmaf(lam, b.y, mu * a.y); pz = fmaf(lam, b.z, mu * a.z);
    const float ux = fmaf(lam, tb.x, mu * ta.x), uy = fmaf(lam, tb.y, mu * ta.y), uz = fmaf(lam, tb.z, mu * ta.z);
    const float inv = rsqrtf(fmaf(uz, uz, fmaf(uy, uy, ux * ux)));
    tx = ux * inv; ty = uy * inv; tz = uz * inv;
}

// the fifth sampled input [R-35]: dv = clamp(v_nom + sigma_v z5, -dv_max, dv_max), z5 = first Box-Muller
// output of the Philox block at counter (k, t + 2^31, iter, b)
template <int MATH>
__device__ __forceinline__ float sample_progress_accel(const DevParams& P, const uint32_t (&rk)[20], uint32_t k,
                                                       uint32_t t, uint32_t iter, uint32_t b, const float vn)
{
    const uint4 r = philox4x32_10(k, t + 0x80000000u, iter, b, rk);
    float a, unused;
    perturb_pair<MATH>(r.x, r.y, P.sigma_v, vn, 0.0f, a, unused);
    return fminf(fmaxf(a, -P.dv_max), P.dv_max);
}

// stage cost of eq.(9) at a pre-step state [R-37]
__device__ __forceinline__ float contour_paper_stage(const DevParams& P, const float4* s_path, const State& x,
                                                     const float theta, const float v_theta, const float4 dT,
                                                     const float dv)
{
    float px, py, pz, tx, ty, tz;
    path_eval(P, s_path, theta, px, py, pz, tx, ty, tz);
    const float ex = x.px - px, ey = x.py - py, ez = x.pz - pz;
    const float e_l = fmaf(ez, tz, fmaf(ey, ty, ex * tx));
    const float e_c2 = fmaxf(fmaf(ez, ez, fmaf(ey, ey, ex * ex)) - e_l * e_l, 0.0f);
    float J = P.q_l * e_l * e_l;
    J = fmaf(P.q_c, e_c2, J);
    J = fmaf(P.w_omega, fmaf(x.oz, x.oz, fmaf(x.oy, x.oy, x.ox * x.ox)), J);
    J = fmaf(P.r_dv, dv * dv, J);
    J = fmaf(P.R, fmaf(dT.w, dT.w, fmaf(dT.z, dT.z, fmaf(dT.y, dT.y, dT.x * dT.x))), J);
    return fmaf(-P.mu, v_theta, J);
}

}  // namespace mppi
