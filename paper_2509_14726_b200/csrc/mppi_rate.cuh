// mppi_rate.cuh -- device functions of the paper's own input model:
// general f_dyn with rotor drag, RK4 on the 17-vector [p, q, v, omega, T], soft body-rate limit.
// Used by the rollout kernel (mppi_rate.cu) and by the plant / nominal-rollout kernels (mppi_kernels.cu).
#pragma once
#include "mppi_device.cuh"
#include "mppi_packed.cuh"

namespace mppi {

struct Deriv { float qw, qx, qy, qz, vx, vy, vz, ox, oy, oz; };     // q slots: 2 q'; p' = v needs no slot

// f_dyn of eq.(2) for the attitude, velocity and body-rate parts at stage state (q, v, o) with rotor
// thrusts T.  Powers of two are kept out of the inner arithmetic (exact rescalings, folded into host
// constants and step sizes): the q slots hold G = 2 q' = q (x) (0, omega); R(q) is formed as its half
// E = R / 2 (diagonal 1/2 - (a^2 + b^2) in two FFMAs, off-diagonals without their factor 2), so
// - R D R^T v = - E (4 D) E^T v with drag4 = 4 D and the thrust term is (2 S / m) e2 with inv_mass2 = 2 / m.
// AXI != 0: the caller has checked drag_x == drag_y (rotor drag of an axisymmetric airframe, as in every
// workload here): R D R^T = d_x R R^T + (d_z - d_x) r3 r3^T, so only the thrust axis r3 = 2 e2 is formed.
// R(q) is the usual polynomial, evaluated at the UN-normalised stage quaternions of RK4 (that is the vector
// field the oracle integrates): with n = |q|^2, u = (qx, qy, qz) it satisfies R R^T v = v + 4 (1 - n)
// [(u . v) u - |u|^2 v] exactly, so
//   v' = [2 S / m - 4 (d_z - d_x) (e2 . v)] e2 + (k |u|^2 - d_x) v - k (u . v) u - g z,   k = 4 d_x (1 - n).
// AXI = 1: stage 1, where q is the step's normalised state (n = 1 to rounding, k dropped): 16 operations;
// AXI = 2: inner stages with the k terms: 29 operations; general form: 43.
// ax, ay, az: torque accelerations tau_i / J_i of the stage's thrusts (J^-1 folded in); c = 2 S / m.
template <int AXI = 0>
__device__ __forceinline__ Deriv fdyn_general(const DevParams& P, const float qw, const float qx, const float qy,
                                              const float qz, const float vx, const float vy, const float vz,
                                              const float ox, const float oy, const float oz, const float ax,
                                              const float ay, const float az, const float c)
{
    Deriv d;
    d.qw = fmaf(-qz, oz, fmaf(-qy, oy, -qx * ox));
    d.qx = fmaf(-qz, oy, fmaf(qy, oz, qw * ox));
    d.qy = fmaf(-qx, oz, fmaf(qz, ox, qw * oy));
    d.qz = fmaf(-qy, ox, fmaf(qx, oy, qw * oz));
    d.ox = fmaf(P.gyx, oy * oz, ax);
    d.oy = fmaf(P.gyy, oz * ox, ay);
    d.oz = fmaf(P.gyz, ox * oy, az);
    if (AXI) {
        const float e2x = fmaf(qx, qz, qw * qy), e2y = fmaf(qy, qz, -qw * qx), e2z = fmaf(-qy, qy, fmaf(-qx, qx, 0.5f));
        const float w = fmaf(-P.drag_dd4, fmaf(e2z, vz, fmaf(e2y, vy, e2x * vx)), c);
        if (AXI == 1) {
            d.vx = fmaf(w, e2x, -P.drag_x * vx);
            d.vy = fmaf(w, e2y, -P.drag_x * vy);
            d.vz = fmaf(w, e2z, fmaf(-P.drag_x, vz, -P.g));
        } else {
            const float uu = fmaf(qz, qz, fmaf(qy, qy, qx * qx));
            const float k = fmaf(-P.drag4_x, fmaf(qw, qw, uu), P.drag4_x);
            const float cu = -k * fmaf(qz, vz, fmaf(qy, vy, qx * vx)), cv = fmaf(k, uu, -P.drag_x);
            d.vx = fmaf(w, e2x, fmaf(cv, vx, cu * qx));
            d.vy = fmaf(w, e2y, fmaf(cv, vy, cu * qy));
            d.vz = fmaf(w, e2z, fmaf(cv, vz, fmaf(cu, qz, -P.g)));
        }
        return d;
    }
    // half columns of R(q): the body axes in the world frame, times 1/2
    const float e0x = fmaf(-qz, qz, fmaf(-qy, qy, 0.5f)), e0y = fmaf(qx, qy, qw * qz), e0z = fmaf(qx, qz, -qw * qy);
    const float e1x = fmaf(qx, qy, -qw * qz), e1y = fmaf(-qz, qz, fmaf(-qx, qx, 0.5f)), e1z = fmaf(qy, qz, qw * qx);
    const float e2x = fmaf(qx, qz, qw * qy), e2y = fmaf(qy, qz, -qw * qx), e2z = fmaf(-qy, qy, fmaf(-qx, qx, 0.5f));
    // - R D R^T v: project v on each body axis, scale by that axis' coefficient [R-30]
    const float b0 = P.drag4_x * fmaf(e0z, vz, fmaf(e0y, vy, e0x * vx));
    const float b1 = P.drag4_y * fmaf(e1z, vz, fmaf(e1y, vy, e1x * vx));
    const float b2 = P.drag4_z * fmaf(e2z, vz, fmaf(e2y, vy, e2x * vx));
    d.vx = fmaf(c, e2x, -fmaf(e2x, b2, fmaf(e1x, b1, e0x * b0)));
    d.vy = fmaf(c, e2y, -fmaf(e2y, b2, fmaf(e1y, b1, e0y * b0)));
    d.vz = fmaf(c, e2z, -fmaf(e2z, b2, fmaf(e1z, b1, e0z * b0))) - P.g;
    return d;
}

// The three thrust combinations the torques of PAPER.md:70 are made of, carried NEXT TO the thrust states:
//   x = (T0 + T1) - (T2 + T3),  y = (T1 - T0) + (T2 - T3),  z = (T2 - T3) - (T1 - T0).
// Each rotor thrust sits near hover (~2 N, ulp 2.4e-7) and collects a rounding error every step; the torques are
// DIFFERENCES of them (~0.1 N), so that error reaches the body rates amplified by lever / J ~ 100: measured at the
// paper's Table I sizes it is what pushed one cost of 8192 beyond rel 1e-4 through the soft body-rate limit
// (profiles/README_r02a.md).  The differences themselves obey D' = the same combination of the rates, so integrating
// them directly keeps their rounding error relative to |D|, ten to twenty times smaller.  They are re-derived from
// the thrusts only when the projection onto [T_min, T_max] actually moved a thrust [R-29].
struct ThrustDiff { float x, y, z; };
__device__ __forceinline__ ThrustDiff thrust_diff(const float4 T)
{
    const float s01 = T.x + T.y, s23 = T.z + T.w, d10 = T.y - T.x, d23 = T.z - T.w;
    return ThrustDiff{s01 - s23, d10 + d23, d23 - d10};
}

// x <- RK4 on the 17-vector [p, q, v, omega, T] with T' = u held over the step; q renormalised; the
// thrust states projected onto [T_min, T_max] afterwards [R-27],[R-29].  D: thrust_diff(T), kept by the caller.
template <bool AXI = false>      // AXI: drag_x == drag_y (see fdyn_general)
__device__ __forceinline__ void rk4_rate_step(const DevParams& P, State& x, float4& T, ThrustDiff& D, const float4 u)
{
    const float h = P.dt, hh = P.h2, hq = P.h4;                       // hq: the q slots of Deriv hold 2 q'
    const float4 Te = make_float4(fmaf(h, u.x, T.x), fmaf(h, u.y, T.y), fmaf(h, u.z, T.z), fmaf(h, u.w, T.w));
    // torque accelerations and collective acceleration of the three distinct stage thrusts T, T + h/2 u, T + h u:
    // linear in the thrusts, so the value at T and the slope along u give all of them
    const ThrustDiff du = thrust_diff(u);
    const float S = (T.x + T.y) + (T.z + T.w), su = (u.x + u.y) + (u.z + u.w);
    const ThrustDiff Dm{fmaf(hh, du.x, D.x), fmaf(hh, du.y, D.y), fmaf(hh, du.z, D.z)};
    const ThrustDiff De{fmaf(h, du.x, D.x), fmaf(h, du.y, D.y), fmaf(h, du.z, D.z)};
    const float a1x = P.ltx * D.x, a1y = P.lty * D.y, a1z = P.ltz * D.z, c1 = S * P.inv_mass2;
    const float amx = P.ltx * Dm.x, amy = P.lty * Dm.y, amz = P.ltz * Dm.z, cm = fmaf(hh, su, S) * P.inv_mass2;
    const float aex = P.ltx * De.x, aey = P.lty * De.y, aez = P.ltz * De.z, ce = fmaf(h, su, S) * P.inv_mass2;
    // stage 1
    Deriv k = fdyn_general<(AXI ? 1 : 0)>(P, x.qw, x.qx, x.qy, x.qz, x.vx, x.vy, x.vz, x.ox, x.oy, x.oz, a1x, a1y, a1z, c1);
    float apx = x.vx, apy = x.vy, apz = x.vz;                         // sums of p' = v over the stages
    Deriv a = k;
    float vx = fmaf(hh, k.vx, x.vx), vy = fmaf(hh, k.vy, x.vy), vz = fmaf(hh, k.vz, x.vz);
    float qw = fmaf(hq, k.qw, x.qw), qx = fmaf(hq, k.qx, x.qx), qy = fmaf(hq, k.qy, x.qy), qz = fmaf(hq, k.qz, x.qz);
    float ox = fmaf(hh, k.ox, x.ox), oy = fmaf(hh, k.oy, x.oy), oz = fmaf(hh, k.oz, x.oz);
#define MPPI_ACC(W)                                                                                    \
    a.qw = fmaf(W, k.qw, a.qw); a.qx = fmaf(W, k.qx, a.qx); a.qy = fmaf(W, k.qy, a.qy); a.qz = fmaf(W, k.qz, a.qz); \
    a.vx = fmaf(W, k.vx, a.vx); a.vy = fmaf(W, k.vy, a.vy); a.vz = fmaf(W, k.vz, a.vz);               \
    a.ox = fmaf(W, k.ox, a.ox); a.oy = fmaf(W, k.oy, a.oy); a.oz = fmaf(W, k.oz, a.oz);
    // stage 2 (state x + h/2 k1, thrusts T + h/2 u)
    apx = fmaf(2.0f, vx, apx); apy = fmaf(2.0f, vy, apy); apz = fmaf(2.0f, vz, apz);
    k = fdyn_general<(AXI ? 2 : 0)>(P, qw, qx, qy, qz, vx, vy, vz, ox, oy, oz, amx, amy, amz, cm);
    MPPI_ACC(2.0f)
    vx = fmaf(hh, k.vx, x.vx); vy = fmaf(hh, k.vy, x.vy); vz = fmaf(hh, k.vz, x.vz);
    qw = fmaf(hq, k.qw, x.qw); qx = fmaf(hq, k.qx, x.qx); qy = fmaf(hq, k.qy, x.qy); qz = fmaf(hq, k.qz, x.qz);
    ox = fmaf(hh, k.ox, x.ox); oy = fmaf(hh, k.oy, x.oy); oz = fmaf(hh, k.oz, x.oz);
    // stage 3
    apx = fmaf(2.0f, vx, apx); apy = fmaf(2.0f, vy, apy); apz = fmaf(2.0f, vz, apz);
    k = fdyn_general<(AXI ? 2 : 0)>(P, qw, qx, qy, qz, vx, vy, vz, ox, oy, oz, amx, amy, amz, cm);
    MPPI_ACC(2.0f)
    vx = fmaf(h, k.vx, x.vx); vy = fmaf(h, k.vy, x.vy); vz = fmaf(h, k.vz, x.vz);
    qw = fmaf(hh, k.qw, x.qw); qx = fmaf(hh, k.qx, x.qx); qy = fmaf(hh, k.qy, x.qy); qz = fmaf(hh, k.qz, x.qz);
    ox = fmaf(h, k.ox, x.ox); oy = fmaf(h, k.oy, x.oy); oz = fmaf(h, k.oz, x.oz);
    // stage 4 (state x + h k3, thrusts T + h u)
    apx += vx; apy += vy; apz += vz;
    k = fdyn_general<(AXI ? 2 : 0)>(P, qw, qx, qy, qz, vx, vy, vz, ox, oy, oz, aex, aey, aez, ce);
    MPPI_ACC(1.0f)
#undef MPPI_ACC
    const float h6 = P.h6;
    x.px = fmaf(h6, apx, x.px); x.py = fmaf(h6, apy, x.py); x.pz = fmaf(h6, apz, x.pz);
    x.vx = fmaf(h6, a.vx, x.vx); x.vy = fmaf(h6, a.vy, x.vy); x.vz = fmaf(h6, a.vz, x.vz);
    x.ox = fmaf(h6, a.ox, x.ox); x.oy = fmaf(h6, a.oy, x.oy); x.oz = fmaf(h6, a.oz, x.oz);
    const float h12 = P.h12;
    const float nw = fmaf(h12, a.qw, x.qw), nx = fmaf(h12, a.qx, x.qx), ny = fmaf(h12, a.qy, x.qy), nz = fmaf(h12, a.qz, x.qz);
    const float inv = rsqrtf(fmaf(nz, nz, fmaf(ny, ny, fmaf(nx, nx, nw * nw))));
    x.qw = nw * inv; x.qx = nx * inv; x.qy = ny * inv; x.qz = nz * inv;
    T.x = fminf(fmaxf(Te.x, P.T_min), P.T_max); T.y = fminf(fmaxf(Te.y, P.T_min), P.T_max);
    T.z = fminf(fmaxf(Te.z, P.T_min), P.T_max); T.w = fminf(fmaxf(Te.w, P.T_min), P.T_max);
    const bool moved = T.x != Te.x || T.y != Te.y || T.z != Te.z || T.w != Te.w;     // the projection acted
    const ThrustDiff Dc = thrust_diff(T);
    D.x = moved ? Dc.x : De.x; D.y = moved ? Dc.y : De.y; D.z = moved ? Dc.z : De.z;
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
    perturb_pair<MATH>(r.x, r.y, P.sigma_v, P.bm_kv, vn, 0.0f, a, unused);
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

// ---- two samples per thread in packed fp32x2 registers (see mppi_packed.cuh): the same model ------------
struct Deriv2 { float2 qw, qx, qy, qz, vx, vy, vz, ox, oy, oz; };

// f_dyn of eq.(2) with drag for two samples; ax, ay, az, c as in fdyn_general (halves = the two samples)
template <int AXI = 0>
__device__ __forceinline__ Deriv2 fdyn_general2(const DevParams& P, const float2 qw, const float2 qx, const float2 qy,
                                                const float2 qz, const float2 vx, const float2 vy, const float2 vz,
                                                const float2 ox, const float2 oy, const float2 oz, const float2 ax,
                                                const float2 ay, const float2 az, const float2 c)
{
    Deriv2 d;                                  // same operations, same order as fdyn_general on each half
    const float2 hf = bc2(0.5f);
    d.qw = fma2(neg2(qz), oz, fma2(neg2(qy), oy, mul2(neg2(qx), ox)));
    d.qx = fma2(neg2(qz), oy, fma2(qy, oz, mul2(qw, ox)));
    d.qy = fma2(neg2(qx), oz, fma2(qz, ox, mul2(qw, oy)));
    d.qz = fma2(neg2(qy), ox, fma2(qx, oy, mul2(qw, oz)));
    d.ox = fma2(P.gyx, mul2(oy, oz), ax);
    d.oy = fma2(P.gyy, mul2(oz, ox), ay);
    d.oz = fma2(P.gyz, mul2(ox, oy), az);
    if (AXI) {
        const float2 e2x = fma2(qx, qz, mul2(qw, qy)), e2y = fma2(qy, qz, mul2(neg2(qw), qx)),
                     e2z = fma2(neg2(qy), qy, fma2(neg2(qx), qx, hf));
        const float2 w = fma2(bc2(-P.drag_dd4), fma2(e2z, vz, fma2(e2y, vy, mul2(e2x, vx))), c);
        const float2 ndx = bc2(-P.drag_x);
        if (AXI == 1) {
            d.vx = fma2(w, e2x, mul2(ndx, vx));
            d.vy = fma2(w, e2y, mul2(ndx, vy));
            d.vz = fma2(w, e2z, fma2(ndx, vz, bc2(-P.g)));
        } else {
            const float2 uu = fma2(qz, qz, fma2(qy, qy, mul2(qx, qx)));
            const float2 k = fma2(bc2(-P.drag4_x), fma2(qw, qw, uu), bc2(P.drag4_x));
            const float2 cu = mul2(neg2(k), fma2(qz, vz, fma2(qy, vy, mul2(qx, vx)))), cv = fma2(k, uu, ndx);
            d.vx = fma2(w, e2x, fma2(cv, vx, mul2(cu, qx)));
            d.vy = fma2(w, e2y, fma2(cv, vy, mul2(cu, qy)));
            d.vz = fma2(w, e2z, fma2(cv, vz, fma2(cu, qz, bc2(-P.g))));
        }
        return d;
    }
    const float2 e0x = fma2(neg2(qz), qz, fma2(neg2(qy), qy, hf)), e0y = fma2(qx, qy, mul2(qw, qz)),
                 e0z = fma2(qx, qz, mul2(neg2(qw), qy));
    const float2 e1x = fma2(qx, qy, mul2(neg2(qw), qz)), e1y = fma2(neg2(qz), qz, fma2(neg2(qx), qx, hf)),
                 e1z = fma2(qy, qz, mul2(qw, qx));
    const float2 e2x = fma2(qx, qz, mul2(qw, qy)), e2y = fma2(qy, qz, mul2(neg2(qw), qx)),
                 e2z = fma2(neg2(qy), qy, fma2(neg2(qx), qx, hf));
    const float2 b0 = mul2(bc2(P.drag4_x), fma2(e0z, vz, fma2(e0y, vy, mul2(e0x, vx))));
    const float2 b1 = mul2(bc2(P.drag4_y), fma2(e1z, vz, fma2(e1y, vy, mul2(e1x, vx))));
    const float2 b2 = mul2(bc2(P.drag4_z), fma2(e2z, vz, fma2(e2y, vy, mul2(e2x, vx))));
    d.vx = fma2(c, e2x, neg2(fma2(e2x, b2, fma2(e1x, b1, mul2(e0x, b0)))));
    d.vy = fma2(c, e2y, neg2(fma2(e2y, b2, fma2(e1y, b1, mul2(e0y, b0)))));
    d.vz = sub2(fma2(c, e2z, neg2(fma2(e2z, b2, fma2(e1z, b1, mul2(e0z, b0))))), bc2(P.g));
    return d;
}

__device__ __forceinline__ float2 clamp2(const float2 v, const float lo, const float hi)
{
    return make_float2(fminf(fmaxf(v.x, lo), hi), fminf(fmaxf(v.y, lo), hi));
}

struct ThrustDiff2 { float2 x, y, z; };
__device__ __forceinline__ ThrustDiff2 thrust_diff2(const float2 T0, const float2 T1, const float2 T2, const float2 T3)
{
    const float2 s01 = add2(T0, T1), s23 = add2(T2, T3), d10 = sub2(T1, T0), d23 = sub2(T2, T3);
    return ThrustDiff2{sub2(s01, s23), add2(d10, d23), sub2(d23, d10)};
}

// rk4_rate_step for two samples: x, T (4 rotor thrust pairs), D (their torque combinations) <- one step with the rates
// ua / ub held; same operations in the same order as rk4_rate_step on each half
template <bool AXI = false>
__device__ __forceinline__ void rk4_rate_step2(const DevParams& P, State2& x, float2 (&T)[4], ThrustDiff2& D, const float4 ua,
                                               const float4 ub)
{
    const float2 h = bc2(P.dt), hh = bc2(P.h2), hq = bc2(P.h4), h6 = bc2(P.h6), h12 = bc2(P.h12), two = bc2(2.0f);
    const float2 u0 = make_float2(ua.x, ub.x), u1 = make_float2(ua.y, ub.y), u2 = make_float2(ua.z, ub.z), u3 = make_float2(ua.w, ub.w);
    const float2 Te0 = fma2(h, u0, T[0]), Te1 = fma2(h, u1, T[1]), Te2 = fma2(h, u2, T[2]), Te3 = fma2(h, u3, T[3]);
    const ThrustDiff2 du = thrust_diff2(u0, u1, u2, u3);
    const float2 S = add2(add2(T[0], T[1]), add2(T[2], T[3])), su = add2(add2(u0, u1), add2(u2, u3));
    const ThrustDiff2 Dm{fma2(hh, du.x, D.x), fma2(hh, du.y, D.y), fma2(hh, du.z, D.z)};
    const ThrustDiff2 De{fma2(h, du.x, D.x), fma2(h, du.y, D.y), fma2(h, du.z, D.z)};
    const float2 ltx = bc2(P.ltx), lty = bc2(P.lty), ltz = bc2(P.ltz), im2 = bc2(P.inv_mass2);
    const float2 a1x = mul2(ltx, D.x), a1y = mul2(lty, D.y), a1z = mul2(ltz, D.z), c1 = mul2(S, im2);
    const float2 amx = mul2(ltx, Dm.x), amy = mul2(lty, Dm.y), amz = mul2(ltz, Dm.z), cm = mul2(fma2(hh, su, S), im2);
    const float2 aex = mul2(ltx, De.x), aey = mul2(lty, De.y), aez = mul2(ltz, De.z), ce = mul2(fma2(h, su, S), im2);
    Deriv2 k = fdyn_general2<(AXI ? 1 : 0)>(P, x.qw, x.qx, x.qy, x.qz, x.vx, x.vy, x.vz, x.ox, x.oy, x.oz, a1x, a1y, a1z, c1);
    float2 apx = x.vx, apy = x.vy, apz = x.vz;
    Deriv2 a = k;
#define MPPI_STAGE2(HS, HQ)                                                                          \
    vx = fma2(HS, k.vx, x.vx); vy = fma2(HS, k.vy, x.vy); vz = fma2(HS, k.vz, x.vz);               \
    qw = fma2(HQ, k.qw, x.qw); qx = fma2(HQ, k.qx, x.qx); qy = fma2(HQ, k.qy, x.qy); qz = fma2(HQ, k.qz, x.qz); \
    ox = fma2(HS, k.ox, x.ox); oy = fma2(HS, k.oy, x.oy); oz = fma2(HS, k.oz, x.oz);
#define MPPI_ACC2(W)                                                                                 \
    a.qw = fma2(W, k.qw, a.qw); a.qx = fma2(W, k.qx, a.qx); a.qy = fma2(W, k.qy, a.qy); a.qz = fma2(W, k.qz, a.qz); \
    a.vx = fma2(W, k.vx, a.vx); a.vy = fma2(W, k.vy, a.vy); a.vz = fma2(W, k.vz, a.vz);             \
    a.ox = fma2(W, k.ox, a.ox); a.oy = fma2(W, k.oy, a.oy); a.oz = fma2(W, k.oz, a.oz);
    float2 vx, vy, vz, qw, qx, qy, qz, ox, oy, oz;
    MPPI_STAGE2(hh, hq)
    apx = fma2(two, vx, apx); apy = fma2(two, vy, apy); apz = fma2(two, vz, apz);
    k = fdyn_general2<(AXI ? 2 : 0)>(P, qw, qx, qy, qz, vx, vy, vz, ox, oy, oz, amx, amy, amz, cm);
    MPPI_ACC2(two)
    MPPI_STAGE2(hh, hq)
    apx = fma2(two, vx, apx); apy = fma2(two, vy, apy); apz = fma2(two, vz, apz);
    k = fdyn_general2<(AXI ? 2 : 0)>(P, qw, qx, qy, qz, vx, vy, vz, ox, oy, oz, amx, amy, amz, cm);
    MPPI_ACC2(two)
    MPPI_STAGE2(h, hh)
    apx = add2(apx, vx); apy = add2(apy, vy); apz = add2(apz, vz);
    k = fdyn_general2<(AXI ? 2 : 0)>(P, qw, qx, qy, qz, vx, vy, vz, ox, oy, oz, aex, aey, aez, ce);
    a.qw = add2(a.qw, k.qw); a.qx = add2(a.qx, k.qx); a.qy = add2(a.qy, k.qy); a.qz = add2(a.qz, k.qz);
    a.vx = add2(a.vx, k.vx); a.vy = add2(a.vy, k.vy); a.vz = add2(a.vz, k.vz);
    a.ox = add2(a.ox, k.ox); a.oy = add2(a.oy, k.oy); a.oz = add2(a.oz, k.oz);
#undef MPPI_STAGE2
#undef MPPI_ACC2
    x.px = fma2(h6, apx, x.px); x.py = fma2(h6, apy, x.py); x.pz = fma2(h6, apz, x.pz);
    x.vx = fma2(h6, a.vx, x.vx); x.vy = fma2(h6, a.vy, x.vy); x.vz = fma2(h6, a.vz, x.vz);
    x.ox = fma2(h6, a.ox, x.ox); x.oy = fma2(h6, a.oy, x.oy); x.oz = fma2(h6, a.oz, x.oz);
    const float2 nw = fma2(h12, a.qw, x.qw), nx = fma2(h12, a.qx, x.qx), ny = fma2(h12, a.qy, x.qy), nz = fma2(h12, a.qz, x.qz);
    const float2 n2 = fma2(nz, nz, fma2(ny, ny, fma2(nx, nx, mul2(nw, nw))));
    const float2 inv = make_float2(rsqrtf(n2.x), rsqrtf(n2.y));
    x.qw = mul2(nw, inv); x.qx = mul2(nx, inv); x.qy = mul2(ny, inv); x.qz = mul2(nz, inv);
    T[0] = clamp2(Te0, P.T_min, P.T_max); T[1] = clamp2(Te1, P.T_min, P.T_max);
    T[2] = clamp2(Te2, P.T_min, P.T_max); T[3] = clamp2(Te3, P.T_min, P.T_max);
    const bool ma = T[0].x != Te0.x || T[1].x != Te1.x || T[2].x != Te2.x || T[3].x != Te3.x;   // the projection acted
    const bool mb = T[0].y != Te0.y || T[1].y != Te1.y || T[2].y != Te2.y || T[3].y != Te3.y;
    const ThrustDiff2 Dc = thrust_diff2(T[0], T[1], T[2], T[3]);
    D.x = make_float2(ma ? Dc.x.x : De.x.x, mb ? Dc.x.y : De.x.y);
    D.y = make_float2(ma ? Dc.y.x : De.y.x, mb ? Dc.y.y : De.y.y);
    D.z = make_float2(ma ? Dc.z.x : De.z.x, mb ? Dc.z.y : De.z.y);
}

}  // namespace mppi
