// mppi_device.cuh -- device-side building blocks of the MPPI hot path (sm_100a, fp32).
//
// Everything here is the product path: it shares no source with oracle/.  Each block cites the
// passage of PAPER.md it implements (readings R-n: DESIGN.md).  One sample lives in one thread;
// the 13-dim state, the cost and the Philox words stay in registers for the whole horizon.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace mppi {

// ---- static per-context constants, passed to every kernel by value (constant bank) ---------
struct DevParams {
    int K, N, B;
    int G, M, P, closed, window;      // gates, reference rows, path points
    int blocks_per_ctrl;               // rollout blocks per controller = K / blockDim.x
    float dt, inv_lambda, sigma, T_min, T_max;
    float inv_mass, g, hover;
    float ltx, lty, ltz;               // (arm/sqrt2)/Jx, (arm/sqrt2)/Jy, c_tau/Jz
    float gyx, gyy, gyz;               // (Jy-Jz)/Jx, (Jz-Jx)/Jy, (Jx-Jy)/Jz   (omega x J omega)
    float w_omega, miss, bonus;        // gate objective constants (BASELINE.json configs[0])
    float Qp, Qv, Qq, Qw, R;           // eq.(8)
    float q_c, q_l, mu, path_L, inv_path_L; // eq.(9) + closed path length
    const float4* gates;               // [G][4]: (c, a_h) (n, a_v) (h, 0) (v = h x n, 0)
    const float4* ref;                 // [M][4]: (p, qw) (qx qy qz, vx) (vy vz, wx wy) (wz,0,0,0)
    const float4* path;                // [P][2]: (P_i, s_i) (t_i, 0)
};

// ---- per-call arguments ---------------------------------------------------------------------
struct StepArgs {
    const float* x0;       // [B][13]
    const int* start;      // [B]
    const float* u_nom;    // [B][N][4]
    float* u_new;          // [B][N][4]
    float* cost;           // [B][K]
    float* weights;        // [B][K]
    float4* du;            // [B][N][K] float4 or nullptr
    float* partials;       // [B][blocks_per_ctrl][4N+4]  (fused pipeline)
    unsigned int* counters;// [B]                         (fused pipeline)
    uint32_t seed_lo, seed_hi, iter;
};

// ---- Philox4x32-10, counter-based (Salmon et al., SC'11) [R-1] -----------------------------
// eq.(3) PAPER.md:78-82 asks for independent Gaussian perturbations; north_star fixes the
// generator and its keying: counter = (sample k, step t, iter, controller b), key = seed.
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        c0 = hi1 ^ c1 ^ k0;
        c1 = lo1;
        c2 = hi0 ^ c3 ^ k1;
        c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return make_uint4(c0, c1, c2, c3);
}

// [R-2] u = (2 (r >> 9) + 1) 2^-24, built without an int->float conversion: the mantissa trick
// gives 1 + (r>>9) 2^-23 in [1,2); subtracting 1 - 2^-24 is exact on this 24-bit lattice.
__device__ __forceinline__ float u01(uint32_t r)
{
    return __uint_as_float(0x3f800000u | (r >> 9)) - 0.99999994f;
}

// [R-3] Box-Muller pair.  MATH = 0: IEEE-accurate library functions.  MATH = 1: MUFU
// approximations (lg2 / rsq / sin / cos), see DESIGN.md "error budget".
template <int MATH>
__device__ __forceinline__ void box_muller(uint32_t ra, uint32_t rb, float& z0, float& z1)
{
    const float u1 = u01(ra), u2 = u01(rb);
    if (MATH == 0) {
        const float rad = sqrtf(-2.0f * logf(u1));
        float s, c;
        sincospif(2.0f * u2, &s, &c);
        z0 = rad * c;
        z1 = rad * s;
    } else {
        // -2 ln u = (-2 ln 2) log2 u
        const float rad = sqrtf(-1.3862943611198906f * __log2f(u1));
        float s, c;
        __sincosf(6.283185307179586f * u2, &s, &c);
        z0 = rad * c;
        z1 = rad * s;
    }
}

// Perturbed, clamped rotor thrusts of one (sample, step) and the perturbation actually applied
// [R-8]: T = clamp(u_nom + sigma z), dU = T - u_nom.
template <int MATH>
__device__ __forceinline__ void sample_thrust(const DevParams& P, uint32_t seed_lo, uint32_t seed_hi,
                                              uint32_t k, uint32_t t, uint32_t iter, uint32_t b,
                                              const float4 un, float4& T, float4& du)
{
    const uint4 r = philox4x32_10(k, t, iter, b, seed_lo, seed_hi);
    float z0, z1, z2, z3;
    box_muller<MATH>(r.x, r.y, z0, z1);
    box_muller<MATH>(r.z, r.w, z2, z3);
    T.x = fminf(fmaxf(fmaf(P.sigma, z0, un.x), P.T_min), P.T_max);
    T.y = fminf(fmaxf(fmaf(P.sigma, z1, un.y), P.T_min), P.T_max);
    T.z = fminf(fmaxf(fmaf(P.sigma, z2, un.z), P.T_min), P.T_max);
    T.w = fminf(fmaxf(fmaf(P.sigma, z3, un.w), P.T_min), P.T_max);
    du = make_float4(T.x - un.x, T.y - un.y, T.z - un.z, T.w - un.w);
}

// ---- quadrotor state and dynamics, eq.(2) PAPER.md:65-72 -------------------------------------
struct State {
    float px, py, pz;
    float qw, qx, qy, qz;
    float vx, vy, vz;
    float ox, oy, oz;
};

// The part of f_dyn that depends on the state: q_dot, v_dot, omega_dot (p_dot = v is used
// directly).  Per-step constants (thrust-derived) are hoisted by the caller:
//   c2 = 2 S/m, cz0 = S/m - g, (ax, ay, az) = J^-1 tau.
struct Deriv { float qw, qx, qy, qz, vx, vy, vz, ox, oy, oz; };

__device__ __forceinline__ Deriv f_dyn(const DevParams& P, float qw, float qx, float qy, float qz,
                                       float ox, float oy, float oz, float c2, float cz0, float ax,
                                       float ay, float az)
{
    Deriv d;
    // q_dot = 1/2 q (x) (0, omega)                              (Hamilton product, body rates)
    d.qw = 0.5f * (-qx * ox - qy * oy - qz * oz);
    d.qx = 0.5f * (qw * ox + qy * oz - qz * oy);
    d.qy = 0.5f * (qw * oy + qz * ox - qx * oz);
    d.qz = 0.5f * (qw * oz + qx * oy - qy * ox);
    // v_dot = g + R(q) [0 0 S]^T / m : third column of R(q)
    d.vx = c2 * (qx * qz + qw * qy);
    d.vy = c2 * (qy * qz - qw * qx);
    d.vz = cz0 - c2 * (qx * qx + qy * qy);
    // omega_dot = J^-1 (tau - omega x J omega), diagonal J
    d.ox = fmaf(P.gyx, oy * oz, ax);
    d.oy = fmaf(P.gyy, oz * ox, ay);
    d.oz = fmaf(P.gyz, ox * oy, az);
    return d;
}

// x <- RK4(f_dyn, x, T, dt), then q <- q / |q|   [R-4],[R-5]; input held over the step.
__device__ __forceinline__ void rk4_step(const DevParams& P, State& x, const float4 T)
{
    const float S = (T.x + T.y) + (T.z + T.w);
    const float c = S * P.inv_mass;
    const float c2 = 2.0f * c, cz0 = c - P.g;
    const float ax = P.ltx * ((T.x + T.y) - (T.z + T.w));     // tau_x / Jx
    const float ay = P.lty * ((T.y + T.z) - (T.x + T.w));     // tau_y / Jy
    const float az = P.ltz * ((T.x + T.z) - (T.y + T.w));     // tau_z / Jz
    const float h = P.dt, h2 = 0.5f * P.dt, h6 = P.dt * (1.0f / 6.0f);

    const Deriv k1 = f_dyn(P, x.qw, x.qx, x.qy, x.qz, x.ox, x.oy, x.oz, c2, cz0, ax, ay, az);
    const float v2x = fmaf(h2, k1.vx, x.vx), v2y = fmaf(h2, k1.vy, x.vy), v2z = fmaf(h2, k1.vz, x.vz);
    const Deriv k2 = f_dyn(P, fmaf(h2, k1.qw, x.qw), fmaf(h2, k1.qx, x.qx), fmaf(h2, k1.qy, x.qy),
                           fmaf(h2, k1.qz, x.qz), fmaf(h2, k1.ox, x.ox), fmaf(h2, k1.oy, x.oy),
                           fmaf(h2, k1.oz, x.oz), c2, cz0, ax, ay, az);
    const float v3x = fmaf(h2, k2.vx, x.vx), v3y = fmaf(h2, k2.vy, x.vy), v3z = fmaf(h2, k2.vz, x.vz);
    const Deriv k3 = f_dyn(P, fmaf(h2, k2.qw, x.qw), fmaf(h2, k2.qx, x.qx), fmaf(h2, k2.qy, x.qy),
                           fmaf(h2, k2.qz, x.qz), fmaf(h2, k2.ox, x.ox), fmaf(h2, k2.oy, x.oy),
                           fmaf(h2, k2.oz, x.oz), c2, cz0, ax, ay, az);
    const float v4x = fmaf(h, k3.vx, x.vx), v4y = fmaf(h, k3.vy, x.vy), v4z = fmaf(h, k3.vz, x.vz);
    const Deriv k4 = f_dyn(P, fmaf(h, k3.qw, x.qw), fmaf(h, k3.qx, x.qx), fmaf(h, k3.qy, x.qy),
                           fmaf(h, k3.qz, x.qz), fmaf(h, k3.ox, x.ox), fmaf(h, k3.oy, x.oy),
                           fmaf(h, k3.oz, x.oz), c2, cz0, ax, ay, az);

    // x + dt/6 (k1 + 2 k2 + 2 k3 + k4); p_dot stage values are v, v2, v3, v4
    x.px = fmaf(h6, (x.vx + v4x) + 2.0f * (v2x + v3x), x.px);
    x.py = fmaf(h6, (x.vy + v4y) + 2.0f * (v2y + v3y), x.py);
    x.pz = fmaf(h6, (x.vz + v4z) + 2.0f * (v2z + v3z), x.pz);
    x.vx = fmaf(h6, (k1.vx + k4.vx) + 2.0f * (k2.vx + k3.vx), x.vx);
    x.vy = fmaf(h6, (k1.vy + k4.vy) + 2.0f * (k2.vy + k3.vy), x.vy);
    x.vz = fmaf(h6, (k1.vz + k4.vz) + 2.0f * (k2.vz + k3.vz), x.vz);
    x.ox = fmaf(h6, (k1.ox + k4.ox) + 2.0f * (k2.ox + k3.ox), x.ox);
    x.oy = fmaf(h6, (k1.oy + k4.oy) + 2.0f * (k2.oy + k3.oy), x.oy);
    x.oz = fmaf(h6, (k1.oz + k4.oz) + 2.0f * (k2.oz + k3.oz), x.oz);
    const float nw = fmaf(h6, (k1.qw + k4.qw) + 2.0f * (k2.qw + k3.qw), x.qw);
    const float nx = fmaf(h6, (k1.qx + k4.qx) + 2.0f * (k2.qx + k3.qx), x.qx);
    const float ny = fmaf(h6, (k1.qy + k4.qy) + 2.0f * (k2.qy + k3.qy), x.qy);
    const float nz = fmaf(h6, (k1.qz + k4.qz) + 2.0f * (k2.qz + k3.qz), x.qz);
    const float inv = rsqrtf(nw * nw + nx * nx + ny * ny + nz * nz);
    x.qw = nw * inv; x.qx = nx * inv; x.qy = ny * inv; x.qz = nz * inv;
}

__device__ __forceinline__ State load_state(const float* __restrict__ x0)
{
    State x;
    x.px = x0[0]; x.py = x0[1]; x.pz = x0[2];
    x.qw = x0[3]; x.qx = x0[4]; x.qy = x0[5]; x.qz = x0[6];
    x.vx = x0[7]; x.vy = x0[8]; x.vz = x0[9];
    x.ox = x0[10]; x.oy = x0[11]; x.oz = x0[12];
    return x;
}

__device__ __forceinline__ int wrap_index(int i, int n)
{
    i %= n;
    return i < 0 ? i + n : i;
}

}  // namespace mppi
