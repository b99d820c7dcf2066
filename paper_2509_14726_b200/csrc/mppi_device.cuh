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
    int pipe_d, pipe_df;               // rollout_pipe_rate_kernel: ring depths in chunks (W / Q rings, F ring)
    int part_stride;                   // floats per partial: 4N + 4 (+ N under OBJ_CONTOUR_PAPER), rounded up to a multiple of 8
    float dt, inv_lambda, sigma, T_min, T_max;
    float bm_k, bm_kv;                 // -2 ln2 sigma^2, -2 ln2 sigma_v^2: Box-Muller radius constants of the fast path
    float h2, h3, h4, h6, h12, hh2, hh3;   // dt/2, dt/3, dt/4, dt/6, dt/12, dt^2/2, dt^2/3
    float inv_mass, g, hover;
    float ltx, lty, ltz;               // (arm/sqrt2)/Jx, (arm/sqrt2)/Jy, c_tau/Jz
    float gyx, gyy, gyz;               // (Jy-Jz)/Jx, (Jz-Jx)/Jy, (Jx-Jy)/Jz   (omega x J omega)
    float w_omega, miss, bonus;        // gate objective constants (BASELINE.json configs[0])
    float q_near, r_near2;             // eq.(7): weight, threshold radius squared [R-24]
    int near_mode;                     // 0: against the step's own target [R-24]; 1: against the horizon's start gate [R-40]
    // the paper's own input model (Table I) [R-27]..[R-32]: u = dT/dt, thrusts are states
    int input_model;
    float rate_max, drag_x, drag_y, drag_z, w_limit, omega_max;
    float drag_dd4;                    // 4 (drag_z - drag_x): axisymmetric form of the drag (drag_x == drag_y)
    float drag4_x, drag4_y, drag4_z, inv_mass2;   // 4 D and 2 / m: fdyn_general works with R / 2 (mppi_rate.cuh)
    float sigma_v, dv_max, v_theta_max, r_dv;   // the paper's own contouring, eq.(9) [R-33]..[R-37]
    float Qp, Qv, Qq, Qw, R;           // eq.(8)
    float q_c, q_l, mu, path_L, inv_path_L; // eq.(9) + closed path length
    const float4* gates;               // [G][4]: (c, a_h) (n, a_v) (h, n.c) (v = h x n, 0)
    const float4* ref;                 // [M][4]: (p, qw) (qx qy qz, vx) (vy vz, wx wy) (wz,0,0,0)
    const float4* path;                // [2][P]: all (P_i, s_i), then all (t_i, 0)
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
    float* partials;       // [B][blocks_per_ctrl][part_stride]: S[4N], 4 spare, [S5[N]]  (fused pipeline)
    float2* headers;       // [B][blocks_per_ctrl]: (m, Z) of every partial, contiguous per controller
    unsigned int* counters;// [B + 1]: last-block tickets per controller, finished controllers (fused pipeline)
    unsigned int* hint;    // [B] or nullptr (fused throughput kernels): written by the combine of one launch, read by
                           // the next: != 0 = many samples carried weight, keep dU in `du` and sum it from there
                           // instead of re-deriving the noise (mppi_rollout.cuh, warp_noise_partial)
    const float* v_nom;    // [B][N] nominal progress accelerations (OBJ_CONTOUR_PAPER), or nullptr
    float* v_new;          // [B][N] updated ones
    const int* prev_front; // [B][N+1] or nullptr: previous-iteration "in front" flags (paper's J_gate, Fig. 2)
    int pdl;               // pipelined kernel only: bit 0 = this launch carries the programmatic-stream-serialization
                           // attribute: do everything that does not depend on the previous kernel in the stream (stage
                           // the track, draw the normals), then griddepcontrol.wait before touching the nominal; bit 1 =
                           // let a dependent launch start once this block's body-rate chain is done (mppi_optimize's chain)
    unsigned int* done_flag;   // mapped host word, or nullptr: set to done_value once every output of the
    unsigned int done_value;   // call is visible to the host (mppi_step_host polls it instead of a stream sync)
#ifdef MPPI_TIMELINE
    unsigned long long* timeline;   // profiling builds only (-DMPPI_TIMELINE): [blocks][16] %globaltimer stamps
#endif
    uint32_t seed_lo, seed_hi, iter;
    uint32_t rk[20];       // Philox round keys: rk[2r] = seed_lo + r W0, rk[2r+1] = seed_hi + r W1
};

// Profiling aid, compiled only with -DMPPI_TIMELINE (never in the library that ships): thread `who` of the block
// stamps %globaltimer into slot i of its block's row.
#ifdef MPPI_TIMELINE
#if MPPI_TIMELINE == 2      // SM-local cycle counter (deltas within one block only)
#define MPPI_STAMP(A, i) do { (A).timeline[(size_t)(blockIdx.y * gridDim.x + blockIdx.x) * 16 + (i)] = (unsigned long long)clock64(); } while (0)
#else
#define MPPI_STAMP(A, i) do { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); \
    (A).timeline[(size_t)(blockIdx.y * gridDim.x + blockIdx.x) * 16 + (i)] = t_; } while (0)
#endif
#else
#define MPPI_STAMP(A, i) do { } while (0)
#endif

// ---- Philox4x32-10, counter-based (Salmon et al., SC'11) [R-1] -----------------------------
// eq.(3) PAPER.md:78-82 asks for independent Gaussian perturbations; north_star fixes the
// generator and its keying: counter = (sample k, step t, iter, controller b), key = seed.
// The ten round keys depend only on the seed: the host puts them in the kernel-argument constant
// bank (StepArgs::rk), so a round is 2 IMAD.WIDE + 2 LOP3 and holds no key registers.
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               const uint32_t (&rk)[20])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        c0 = hi1 ^ c1 ^ rk[2 * r];
        c1 = lo1;
        c2 = hi0 ^ c3 ^ rk[2 * r + 1];
        c3 = lo0;
    }
    return make_uint4(c0, c1, c2, c3);
}

// [R-2] u = (2 (r >> 9) + 1) 2^-24, built without an int->float conversion: the mantissa trick
// gives 1 + (r>>9) 2^-23 in [1,2); subtracting 1 - 2^-24 is exact on this 24-bit lattice.
__device__ __forceinline__ float u01(uint32_t r)
{
    return __uint_as_float(0x3f800000u | (r >> 9)) - 0.99999994f;
}

// MUFU approximations with flush-to-zero forms (no denormal fix-up code: every argument below is a
// normal number by construction).
__device__ __forceinline__ float mufu_lg2(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_rsq(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_sqrt(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_sin(float x) { float y; asm("sin.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_cos(float x) { float y; asm("cos.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_ex2(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// [R-3] Box-Muller pair scaled by sigma, added to the nominal: (a, b) = (una, unb) + sigma (z0, z1),
// z0 = rad cos(2 pi u2), z1 = rad sin(2 pi u2), rad = sqrt(-2 ln u1).
// MATH = 0: IEEE-accurate library functions, in the oracle's operation order.
// MATH = 1: MUFU lg2 / rsq / sin / cos.  The angle is taken as 2 pi (u2 - 1/2) in [-pi, pi), where the
// MUFU error bound holds, and the sign flip cos(x - pi) = -cos x is folded into the final fma.
// The pair in two halves, so that the pipelined kernel can draw the state-independent part (Philox, radius, angle)
// before the nominal is known: perturb_pair = perturb_finish(perturb_prepare), operation for operation.
//   MATH = 0: f0 = rad cos, f1 = rad sin          -> a = fma(sigma, f0, una)
//   MATH = 1: f0 = sigma rad, f1 = angle          -> a = fma(-f0, MUFU.COS(f1), una)
template <int MATH>
__device__ __forceinline__ void perturb_prepare(uint32_t ra, uint32_t rb, float bm_k, float& f0, float& f1)
{
    if (MATH == 0) {
        const float u1 = u01(ra), u2 = u01(rb);
        const float rad = sqrtf(-2.0f * logf(u1));
        float s, c;
        sincospif(2.0f * u2, &s, &c);
        f0 = rad * c;
        f1 = rad * s;
    } else {
        // rad = sigma sqrt(-2 ln u1) = sqrt(bm_k lg2 u1), bm_k = -2 ln2 sigma^2 from the host: one multiply
        // and MUFU.SQRT.
        f0 = mufu_sqrt(mufu_lg2(u01(ra)) * bm_k);
        // ang = 2 pi (u2 - 1/2) = 2 pi m2 - 3 pi + 2 pi 2^-24 with m2 = 1 + (rb >> 9) 2^-23 in [1, 2): ONE fma
        // straight from the mantissa trick.  The additive constant is the float next to
        // -3 pi + 2 pi 2^-24 - 1.5 (fl(2 pi) - 2 pi), which centres the error of fl(2 pi) m2 on m2 = 1.5:
        // |angle error| <= 3.4e-7 rad, below the MUFU.SIN / MUFU.COS error itself.
        const float m2 = __uint_as_float(0x3f800000u | (rb >> 9));
        f1 = fmaf(m2, 6.283185307179586f, -9.42477798461914f);
    }
}
template <int MATH>
__device__ __forceinline__ void perturb_finish(float f0, float f1, float sigma, float una, float unb, float& a, float& b)
{
    if (MATH == 0) {
        a = fmaf(sigma, f0, una);
        b = fmaf(sigma, f1, unb);
    } else {
        a = fmaf(-f0, mufu_cos(f1), una);
        b = fmaf(-f0, mufu_sin(f1), unb);
    }
}
template <int MATH>
__device__ __forceinline__ void perturb_pair(uint32_t ra, uint32_t rb, float sigma, float bm_k, float una, float unb,
                                             float& a, float& b)
{
    float f0, f1;
    perturb_prepare<MATH>(ra, rb, bm_k, f0, f1);
    perturb_finish<MATH>(f0, f1, sigma, una, unb, a, b);
}

// Perturbed, clamped rotor thrusts of one (sample, step) [R-8]: T = clamp(u_nom + sigma z).
// The perturbation actually applied is dU = T - u_nom (formed by the callers that need it).
template <int MATH>
__device__ __forceinline__ float4 sample_input(const DevParams& P, const uint32_t (&rk)[20], uint32_t k,
                                               uint32_t t, uint32_t iter, uint32_t b, const float4 un,
                                               const float lo, const float hi)
{
    const uint4 r = philox4x32_10(k, t, iter, b, rk);
    float4 T;
    perturb_pair<MATH>(r.x, r.y, P.sigma, P.bm_k, un.x, un.y, T.x, T.y);
    perturb_pair<MATH>(r.z, r.w, P.sigma, P.bm_k, un.z, un.w, T.z, T.w);
    T.x = fminf(fmaxf(T.x, lo), hi);
    T.y = fminf(fmaxf(T.y, lo), hi);
    T.z = fminf(fmaxf(T.z, lo), hi);
    T.w = fminf(fmaxf(T.w, lo), hi);
    return T;
}
template <int MATH>
__device__ __forceinline__ float4 sample_thrust(const DevParams& P, const uint32_t (&rk)[20], uint32_t k,
                                                uint32_t t, uint32_t iter, uint32_t b, const float4 un)
{
    return sample_input<MATH>(P, rk, k, t, iter, b, un, P.T_min, P.T_max);
}

// ---- quadrotor state and dynamics, eq.(2) PAPER.md:65-72 -------------------------------------
struct State {
    float px, py, pz;
    float qw, qx, qy, qz;
    float vx, vy, vz;
    float ox, oy, oz;
};

// x <- RK4(f_dyn, x, T, dt), then q <- q / |q|   [R-4],[R-5]; input held over the step.
//
// f_dyn (eq.(2)) has a triangular structure that the step exploits to cut the instruction count:
//   omega_dot depends on omega only           -> its four stages form their own chain
//   q_dot = 1/2 G(q, omega), G = q (x) (0,w)  -> the 1/2 is folded into the step constants
//   v_dot = (c2 r_x, c2 r_y, cz0 - c2 r_z), r(q) = (qx qz + qw qy, qy qz - qw qx, qx^2 + qy^2),
//           c2 = 2 S/m, cz0 = S/m - g         -> only r(q_i) is evaluated per stage
//   p_dot = v                                 -> p_new = p + h v + h^2/6 (a1 + a2 + a3),
//                                                v_new = v + h/6 (a1 + 2 a2 + 2 a3 + a4)
// which is the classical RK4 written out (the v stages never need to be formed).
__device__ __forceinline__ void rk4_step(const DevParams& P, State& x, const float4 T)
{
    const float s01 = T.x + T.y, s23 = T.z + T.w;
    const float c = (s01 + s23) * P.inv_mass;                  // S / m
    const float ax = P.ltx * (s01 - s23);                      // tau_x / Jx
    const float d10 = T.y - T.x, d23 = T.z - T.w;
    const float ay = P.lty * (d10 + d23);                      // tau_y / Jy  ((T1 + T2) - (T0 + T3))
    const float az = P.ltz * (d23 - d10);                      // tau_z / Jz  ((T0 + T2) - (T1 + T3))
    const float cz0 = c - P.g;
    const float kp = c * P.hh3, kv = c * P.h3;                 // h^2/6 c2, h/6 c2

    // ---- stage 1 (state x)
    float kox = fmaf(P.gyx, x.oy * x.oz, ax), koy = fmaf(P.gyy, x.oz * x.ox, ay), koz = fmaf(P.gyz, x.ox * x.oy, az);
    float gw = fmaf(-x.qz, x.oz, fmaf(-x.qy, x.oy, -x.qx * x.ox));
    float gx = fmaf(-x.qz, x.oy, fmaf(x.qy, x.oz, x.qw * x.ox));
    float gy = fmaf(-x.qx, x.oz, fmaf(x.qz, x.ox, x.qw * x.oy));
    float gz = fmaf(-x.qy, x.ox, fmaf(x.qx, x.oy, x.qw * x.oz));
    const float r1x = fmaf(x.qw, x.qy, x.qx * x.qz), r1y = fmaf(-x.qw, x.qx, x.qy * x.qz),
                r1z = fmaf(x.qy, x.qy, x.qx * x.qx);
    float no_x = fmaf(P.h6, kox, x.ox), no_y = fmaf(P.h6, koy, x.oy), no_z = fmaf(P.h6, koz, x.oz);
    float nw = fmaf(P.h12, gw, x.qw), nx = fmaf(P.h12, gx, x.qx), ny = fmaf(P.h12, gy, x.qy), nz = fmaf(P.h12, gz, x.qz);
    float ox = fmaf(P.h2, kox, x.ox), oy = fmaf(P.h2, koy, x.oy), oz = fmaf(P.h2, koz, x.oz);
    float qw = fmaf(P.h4, gw, x.qw), qx = fmaf(P.h4, gx, x.qx), qy = fmaf(P.h4, gy, x.qy), qz = fmaf(P.h4, gz, x.qz);

    // ---- stage 2
    kox = fmaf(P.gyx, oy * oz, ax); koy = fmaf(P.gyy, oz * ox, ay); koz = fmaf(P.gyz, ox * oy, az);
    gw = fmaf(-qz, oz, fmaf(-qy, oy, -qx * ox));
    gx = fmaf(-qz, oy, fmaf(qy, oz, qw * ox));
    gy = fmaf(-qx, oz, fmaf(qz, ox, qw * oy));
    gz = fmaf(-qy, ox, fmaf(qx, oy, qw * oz));
    const float r2x = fmaf(qw, qy, qx * qz), r2y = fmaf(-qw, qx, qy * qz), r2z = fmaf(qy, qy, qx * qx);
    no_x = fmaf(P.h3, kox, no_x); no_y = fmaf(P.h3, koy, no_y); no_z = fmaf(P.h3, koz, no_z);
    nw = fmaf(P.h6, gw, nw); nx = fmaf(P.h6, gx, nx); ny = fmaf(P.h6, gy, ny); nz = fmaf(P.h6, gz, nz);
    ox = fmaf(P.h2, kox, x.ox); oy = fmaf(P.h2, koy, x.oy); oz = fmaf(P.h2, koz, x.oz);
    qw = fmaf(P.h4, gw, x.qw); qx = fmaf(P.h4, gx, x.qx); qy = fmaf(P.h4, gy, x.qy); qz = fmaf(P.h4, gz, x.qz);

    // ---- stage 3
    kox = fmaf(P.gyx, oy * oz, ax); koy = fmaf(P.gyy, oz * ox, ay); koz = fmaf(P.gyz, ox * oy, az);
    gw = fmaf(-qz, oz, fmaf(-qy, oy, -qx * ox));
    gx = fmaf(-qz, oy, fmaf(qy, oz, qw * ox));
    gy = fmaf(-qx, oz, fmaf(qz, ox, qw * oy));
    gz = fmaf(-qy, ox, fmaf(qx, oy, qw * oz));
    const float r3x = fmaf(qw, qy, qx * qz), r3y = fmaf(-qw, qx, qy * qz), r3z = fmaf(qy, qy, qx * qx);
    no_x = fmaf(P.h3, kox, no_x); no_y = fmaf(P.h3, koy, no_y); no_z = fmaf(P.h3, koz, no_z);
    nw = fmaf(P.h6, gw, nw); nx = fmaf(P.h6, gx, nx); ny = fmaf(P.h6, gy, ny); nz = fmaf(P.h6, gz, nz);
    ox = fmaf(P.dt, kox, x.ox); oy = fmaf(P.dt, koy, x.oy); oz = fmaf(P.dt, koz, x.oz);
    qw = fmaf(P.h2, gw, x.qw); qx = fmaf(P.h2, gx, x.qx); qy = fmaf(P.h2, gy, x.qy); qz = fmaf(P.h2, gz, x.qz);

    // ---- stage 4
    kox = fmaf(P.gyx, oy * oz, ax); koy = fmaf(P.gyy, oz * ox, ay); koz = fmaf(P.gyz, ox * oy, az);
    gw = fmaf(-qz, oz, fmaf(-qy, oy, -qx * ox));
    gx = fmaf(-qz, oy, fmaf(qy, oz, qw * ox));
    gy = fmaf(-qx, oz, fmaf(qz, ox, qw * oy));
    gz = fmaf(-qy, ox, fmaf(qx, oy, qw * oz));
    const float r4x = fmaf(qw, qy, qx * qz), r4y = fmaf(-qw, qx, qy * qz), r4z = fmaf(qy, qy, qx * qx);
    x.ox = fmaf(P.h6, kox, no_x); x.oy = fmaf(P.h6, koy, no_y); x.oz = fmaf(P.h6, koz, no_z);
    nw = fmaf(P.h12, gw, nw); nx = fmaf(P.h12, gx, nx); ny = fmaf(P.h12, gy, ny); nz = fmaf(P.h12, gz, nz);

    // ---- translation: A = r1 + r2 + r3, Bv = r1 + 2 r2 + 2 r3 + r4
    const float mx = r2x + r3x, my = r2y + r3y, mz = r2z + r3z;
    const float Ax = r1x + mx, Ay = r1y + my, Az = r1z + mz;
    x.px = fmaf(kp, Ax, fmaf(P.dt, x.vx, x.px));
    x.py = fmaf(kp, Ay, fmaf(P.dt, x.vy, x.py));
    x.pz = fmaf(-kp, Az, fmaf(P.hh2, cz0, fmaf(P.dt, x.vz, x.pz)));
    x.vx = fmaf(kv, (Ax + mx) + r4x, x.vx);
    x.vy = fmaf(kv, (Ay + my) + r4y, x.vy);
    x.vz = fmaf(-kv, (Az + mz) + r4z, fmaf(P.dt, cz0, x.vz));

    // ---- renormalise once per step [R-5]
    const float inv = rsqrtf(fmaf(nz, nz, fmaf(ny, ny, fmaf(nx, nx, nw * nw))));
    x.qw = nw * inv; x.qx = nx * inv; x.qy = ny * inv; x.qz = nz * inv;
}

// A rollout whose cost is not representable in fp32 -- NaN, or beyond the range: a diverged sample (large noise on a
// long horizon, Inf - Inf inside the dynamics) -- counts as cost kCostCap: weight exactly 0 unless every sample of
// the controller diverged (then they all weigh the same and the update stays finite).  Without this one such sample
// poisons the controller: fminf drops the NaN from the minimum, exp(m - NaN) puts it into Z and from there into every
// weight and every entry of u_new.  [R-41]; the oracle applies the same cap.
constexpr float kCostCap = 3.0e38f;
__device__ __forceinline__ float sanitize_cost(const float J) { return fabsf(J) <= kCostCap ? J : kCostCap; }

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
