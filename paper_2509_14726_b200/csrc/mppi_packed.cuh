// mppi_packed.cuh -- two samples per thread in packed fp32x2 registers (sm_100a FFMA2 / FMUL2 / FADD2).
//
// Blackwell's FMA pipe executes `fma.rn.f32x2` on a 64-bit register pair at the same per-lane rate as
// scalar FFMA but with ONE issue slot and ONE set of operand reads for two results.  The scalar
// rollout is bound by exactly those two resources (profiles/README_r01.md: issue slots 78 %, dispatch
// and math-pipe-throttle stalls), so the throughput variant carries sample 2j in the .x halves and
// sample 2j+1 in the .y halves of every state register.  Each half performs the same operations in
// the same order as the scalar `rk4_step`, so the two variants agree bit for bit.
#pragma once
#include "mppi_device.cuh"

namespace mppi {

struct State2 {
    float2 px, py, pz;
    float2 qw, qx, qy, qz;
    float2 vx, vy, vz;
    float2 ox, oy, oz;
};

__device__ __forceinline__ float2 bc2(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }   // folds into the operand modifier
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { return __fadd2_rn(a, neg2(b)); }
__device__ __forceinline__ float2 fma2(float a, float2 b, float2 c) { return __ffma2_rn(bc2(a), b, c); }

__device__ __forceinline__ State2 splat_state(const State& s)
{
    State2 x;
    x.px = bc2(s.px); x.py = bc2(s.py); x.pz = bc2(s.pz);
    x.qw = bc2(s.qw); x.qx = bc2(s.qx); x.qy = bc2(s.qy); x.qz = bc2(s.qz);
    x.vx = bc2(s.vx); x.vy = bc2(s.vy); x.vz = bc2(s.vz);
    x.ox = bc2(s.ox); x.oy = bc2(s.oy); x.oz = bc2(s.oz);
    return x;
}

template <int H>
__device__ __forceinline__ float half_of(float2 v) { return H == 0 ? v.x : v.y; }

// scalar view of one half (register aliasing: no instructions)
template <int H>
__device__ __forceinline__ State lane_state(const State2& s)
{
    State x;
    x.px = half_of<H>(s.px); x.py = half_of<H>(s.py); x.pz = half_of<H>(s.pz);
    x.qw = half_of<H>(s.qw); x.qx = half_of<H>(s.qx); x.qy = half_of<H>(s.qy); x.qz = half_of<H>(s.qz);
    x.vx = half_of<H>(s.vx); x.vy = half_of<H>(s.vy); x.vz = half_of<H>(s.vz);
    x.ox = half_of<H>(s.ox); x.oy = half_of<H>(s.oy); x.oz = half_of<H>(s.oz);
    return x;
}

// x <- RK4(f_dyn, x, T, dt), q <- q/|q| for two samples; Ta / Tb are their clamped rotor thrusts.
// Same formulation as rk4_step (mppi_device.cuh): eq.(2), [R-4], [R-5].
// SYMZ: the caller has checked P.gyz == 0 (Jx == Jy, the usual symmetric airframe and every config of
// BASELINE.json): fma(0, ox oy, az) is az bit for bit, so the yaw-rate derivative of all four stages is
// the constant az and its eight multiply-adds (and the third-stage yaw rate, equal to the second) drop
// out with results identical to the general form.
template <bool SYMZ>
__device__ __forceinline__ void rk4_step2(const DevParams& P, State2& x, const float4 Ta, const float4 Tb)
{
    const float2 T0 = make_float2(Ta.x, Tb.x), T1 = make_float2(Ta.y, Tb.y), T2 = make_float2(Ta.z, Tb.z),
                 T3 = make_float2(Ta.w, Tb.w);
    const float2 s01 = add2(T0, T1), s23 = add2(T2, T3);
    const float2 c = mul2(add2(s01, s23), bc2(P.inv_mass));                    // S / m
    const float2 ax = mul2(bc2(P.ltx), sub2(s01, s23));                        // tau_x / Jx
    const float2 d10 = sub2(T1, T0), d23 = sub2(T2, T3);
    const float2 ay = mul2(bc2(P.lty), add2(d10, d23));                        // tau_y / Jy
    const float2 az = mul2(bc2(P.ltz), sub2(d23, d10));                        // tau_z / Jz
    const float2 cz0 = sub2(c, bc2(P.g));
    const float2 kp = mul2(c, bc2(P.hh3)), kv = mul2(c, bc2(P.h3));

#define MPPI_STAGE_DERIV(OX, OY, OZ, QW, QX, QY, QZ)                                        \
    kox = fma2(P.gyx, mul2(OY, OZ), ax); koy = fma2(P.gyy, mul2(OZ, OX), ay);              \
    koz = SYMZ ? az : fma2(P.gyz, mul2(OX, OY), az);                                         \
    gw = fma2(neg2(QZ), OZ, fma2(neg2(QY), OY, mul2(neg2(QX), OX)));                         \
    gx = fma2(neg2(QZ), OY, fma2(QY, OZ, mul2(QW, OX)));                                     \
    gy = fma2(neg2(QX), OZ, fma2(QZ, OX, mul2(QW, OY)));                                     \
    gz = fma2(neg2(QY), OX, fma2(QX, OY, mul2(QW, OZ)));

    float2 kox, koy, koz, gw, gx, gy, gz;
    // ---- stage 1 (state x)
    MPPI_STAGE_DERIV(x.ox, x.oy, x.oz, x.qw, x.qx, x.qy, x.qz)
    const float2 r1x = fma2(x.qw, x.qy, mul2(x.qx, x.qz)), r1y = fma2(neg2(x.qw), x.qx, mul2(x.qy, x.qz)),
                 r1z = fma2(x.qy, x.qy, mul2(x.qx, x.qx));
    float2 no_x = fma2(P.h6, kox, x.ox), no_y = fma2(P.h6, koy, x.oy), no_z = fma2(P.h6, koz, x.oz);
    float2 nw = fma2(P.h12, gw, x.qw), nx = fma2(P.h12, gx, x.qx), ny = fma2(P.h12, gy, x.qy), nz = fma2(P.h12, gz, x.qz);
    float2 ox = fma2(P.h2, kox, x.ox), oy = fma2(P.h2, koy, x.oy), oz = fma2(P.h2, koz, x.oz);
    float2 qw = fma2(P.h4, gw, x.qw), qx = fma2(P.h4, gx, x.qx), qy = fma2(P.h4, gy, x.qy), qz = fma2(P.h4, gz, x.qz);

    // ---- stage 2
    MPPI_STAGE_DERIV(ox, oy, oz, qw, qx, qy, qz)
    const float2 r2x = fma2(qw, qy, mul2(qx, qz)), r2y = fma2(neg2(qw), qx, mul2(qy, qz)), r2z = fma2(qy, qy, mul2(qx, qx));
    no_x = fma2(P.h3, kox, no_x); no_y = fma2(P.h3, koy, no_y); no_z = fma2(P.h3, koz, no_z);
    nw = fma2(P.h6, gw, nw); nx = fma2(P.h6, gx, nx); ny = fma2(P.h6, gy, ny); nz = fma2(P.h6, gz, nz);
    ox = fma2(P.h2, kox, x.ox); oy = fma2(P.h2, koy, x.oy); oz = fma2(P.h2, koz, x.oz);
    qw = fma2(P.h4, gw, x.qw); qx = fma2(P.h4, gx, x.qx); qy = fma2(P.h4, gy, x.qy); qz = fma2(P.h4, gz, x.qz);

    // ---- stage 3
    MPPI_STAGE_DERIV(ox, oy, oz, qw, qx, qy, qz)
    const float2 r3x = fma2(qw, qy, mul2(qx, qz)), r3y = fma2(neg2(qw), qx, mul2(qy, qz)), r3z = fma2(qy, qy, mul2(qx, qx));
    no_x = fma2(P.h3, kox, no_x); no_y = fma2(P.h3, koy, no_y); no_z = fma2(P.h3, koz, no_z);
    nw = fma2(P.h6, gw, nw); nx = fma2(P.h6, gx, nx); ny = fma2(P.h6, gy, ny); nz = fma2(P.h6, gz, nz);
    ox = fma2(P.dt, kox, x.ox); oy = fma2(P.dt, koy, x.oy); oz = fma2(P.dt, koz, x.oz);
    qw = fma2(P.h2, gw, x.qw); qx = fma2(P.h2, gx, x.qx); qy = fma2(P.h2, gy, x.qy); qz = fma2(P.h2, gz, x.qz);

    // ---- stage 4
    MPPI_STAGE_DERIV(ox, oy, oz, qw, qx, qy, qz)
    const float2 r4x = fma2(qw, qy, mul2(qx, qz)), r4y = fma2(neg2(qw), qx, mul2(qy, qz)), r4z = fma2(qy, qy, mul2(qx, qx));
    x.ox = fma2(P.h6, kox, no_x); x.oy = fma2(P.h6, koy, no_y); x.oz = fma2(P.h6, koz, no_z);
    nw = fma2(P.h12, gw, nw); nx = fma2(P.h12, gx, nx); ny = fma2(P.h12, gy, ny); nz = fma2(P.h12, gz, nz);
#undef MPPI_STAGE_DERIV

    // ---- translation: A = r1 + r2 + r3, Bv = r1 + 2 r2 + 2 r3 + r4
    const float2 mx = add2(r2x, r3x), my = add2(r2y, r3y), mz = add2(r2z, r3z);
    const float2 Ax = add2(r1x, mx), Ay = add2(r1y, my), Az = add2(r1z, mz);
    x.px = fma2(kp, Ax, fma2(P.dt, x.vx, x.px));
    x.py = fma2(kp, Ay, fma2(P.dt, x.vy, x.py));
    x.pz = fma2(neg2(kp), Az, fma2(P.hh2, cz0, fma2(P.dt, x.vz, x.pz)));
    x.vx = fma2(kv, add2(add2(Ax, mx), r4x), x.vx);
    x.vy = fma2(kv, add2(add2(Ay, my), r4y), x.vy);
    x.vz = fma2(neg2(kv), add2(add2(Az, mz), r4z), fma2(P.dt, cz0, x.vz));

    // ---- renormalise once per step [R-5]
    const float2 n2 = fma2(nz, nz, fma2(ny, ny, fma2(nx, nx, mul2(nw, nw))));
    const float2 inv = make_float2(rsqrtf(n2.x), rsqrtf(n2.y));
    x.qw = mul2(nw, inv); x.qx = mul2(nx, inv); x.qy = mul2(ny, inv); x.qz = mul2(nz, inv);
}

}  // namespace mppi
