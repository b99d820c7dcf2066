// mppi_scan.cuh -- the time-parallel latency kernel: one rollout split over SIXTEEN LANES ALONG THE HORIZON.
//
// For a lone controller the iteration time of every other kernel here is the dependent chain of N RK4 steps
// (configs[1]: 50 steps x ~200 cycles even with the chain cut into three pipelined roles, mppi_pipe.cuh).  Under
// the thrust-input model with a symmetric airframe (Jx == Jy; every configuration of BASELINE.json) eq.(2)
// is a CASCADE OF LINEAR RECURRENCES once the thrusts are drawn, and linear recurrences are
// associative scans:
//
//   omega_z     omega_z' = tau_z / Jz                               a prefix sum
//   omega_xy    w = omega_x + i omega_y:  w' = i kappa omega_z(t) w + (tau_x/Jx + i tau_y/Jy), kappa = (Jz - Jx)/Jx:
//               one RK4 step is the complex affine map w -> H_t w + p_t         a scan of affine maps
//   q           q' = 1/2 q (x) (0, omega): one RK4 step is q -> q (x) m_t(omega), and the per-step renormalisation
//               [R-5] is a scalar, so it commutes with the products               a scan of quaternion products
//   v, p        v' = (S/m) R(q) e3 - g e3,  p' = v: sums                          two prefix sums
//
// So lane c of a sample's 16 lanes owns the steps [c L, (c + 1) L), L = ceil(N / 16) <= 4.  It draws their thrusts,
// runs its chunk of each recurrence from a neutral start (omega_xy: homogeneous + particular solution; attitude:
// from the identity quaternion, in the chunk's own frame), the chunks are joined by warp-shuffle scans over the 16
// lanes, and the chunk-frame results are carried into the world frame by the chunk's start attitude:
//     R(q_s (x) l) = R(q_s) R(l)   for the polynomial R(q) v = q v q*, so with  rho_i = 1/2 R(l_i) e3  (l_i the
//     chunk-frame stage quaternion) and  eps_i = 1/2 (1 - |l_i|^2)  the stage accelerations of rk4_step are
//     v'_i = (2 S/m) (R(q_s) rho_i + eps_i e3) - g e3   -- eps_i carries the "1 - 2 (qx^2 + qy^2)" of eq.(2)'s R(q)
//     at the UN-normalised stage quaternions, where |q_i|^2 != 1 (left out it costs 1e-3 of the thrust acceleration).
// The arithmetic is the same RK4 with the same per-step renormalisation as rk4_step in another association order:
// the states agree with it to rounding (not bit for bit), and parity is against the float64 oracle as for every kernel.
//
// The gate objective (configs[0], [1], [4]) is a state machine along the horizon (target switching),
// but its only state across a chunk boundary is the target index: every lane scores its chunk under a hypothesis for
// it, the first lane (in horizon order) whose chunk switches the target fixes the hypothesis of all later lanes, and
// those are re-scored -- one round per chunk that contains a valid pass, plus one.  Same decisions as GateCost::step.
//
// Block = 16 lanes x up to 32 samples (warp w: samples 2w, 2w + 1; 512 threads at most); grid = (ceil(K / samples), B),
// one block per SM; the host takes fewer samples per block when that lets a lone controller cover every SM
// (configs[1]: 147 blocks of 28 samples on 148 SMs).
// The fused update needs no re-derivation of the noise: every lane still holds the thrusts of its steps.
#pragma once
#include "mppi_rollout.cuh"

namespace mppi {

constexpr int kScanC = 16;                 // lanes per sample = chunks of the horizon
constexpr int kScanL = 4;                  // steps per chunk at most: N <= kScanC * kScanL = 64
constexpr int kScanSamples = 32;           // samples per block at most (the host may take fewer, even, >= kScanMinSamples,
constexpr int kScanMinSamples = 8;         // so that a lone controller's blocks cover every SM): blockDim.x = 16 x samples
constexpr int kScanThreads = kScanSamples * kScanC;
constexpr int kScanMaxN = kScanC * kScanL;

// float4 units of dynamic shared memory after the nominal + track + 16 float4 of reduction scratch
__host__ __device__ inline size_t scan_extra_f4(int N, int nb, int spb)
{
    return (size_t)(spb / 2) * N                // s_acc [warps][N]: weighted perturbations / combine scratch
           + 8                                  // s_cost [32]
           + (size_t)(3 * nb + 3) / 4;          // combine scratch
}

__device__ __forceinline__ float up16(const float v, const int d) { return __shfl_up_sync(kFull, v, d, kScanC); }

// one RK4 step of (omega_x, omega_y) given the three distinct stage values of omega_z (stage 2 and 3 share theirs),
// in the operation order of rk4_step (gyz == 0: the yaw rate has a constant derivative)
__device__ __forceinline__ void omega_xy_step(const DevParams& P, float& ox, float& oy, const float ax, const float ay,
                                              const float z1, const float z2, const float z4)
{
    float kx = fmaf(P.gyx, oy * z1, ax), ky = fmaf(P.gyy, z1 * ox, ay);
    float nx = fmaf(P.h6, kx, ox), ny = fmaf(P.h6, ky, oy);
    float sx = fmaf(P.h2, kx, ox), sy = fmaf(P.h2, ky, oy);
    kx = fmaf(P.gyx, sy * z2, ax); ky = fmaf(P.gyy, z2 * sx, ay);
    nx = fmaf(P.h3, kx, nx); ny = fmaf(P.h3, ky, ny);
    sx = fmaf(P.h2, kx, ox); sy = fmaf(P.h2, ky, oy);
    kx = fmaf(P.gyx, sy * z2, ax); ky = fmaf(P.gyy, z2 * sx, ay);
    nx = fmaf(P.h3, kx, nx); ny = fmaf(P.h3, ky, ny);
    sx = fmaf(P.dt, kx, ox); sy = fmaf(P.dt, ky, oy);
    kx = fmaf(P.gyx, sy * z4, ax); ky = fmaf(P.gyy, z4 * sx, ay);
    ox = fmaf(P.h6, kx, nx); oy = fmaf(P.h6, ky, ny);
}

// quaternion rate times two: G(q, w) = q (x) (0, w)
#define MPPI_SG(QW, QX, QY, QZ, OX, OY, OZ, GW, GX, GY, GZ)                \
    GW = fmaf(-(QZ), OZ, fmaf(-(QY), OY, -(QX) * (OX)));                   \
    GX = fmaf(-(QZ), OY, fmaf(QY, OZ, (QW) * (OX)));                       \
    GY = fmaf(-(QX), OZ, fmaf(QZ, OX, (QW) * (OY)));                       \
    GZ = fmaf(-(QY), OX, fmaf(QX, OY, (QW) * (OZ)));
// chunk-frame thrust direction of a stage quaternion: rho = 1/2 R(l) e3, eps = 1/2 (1 - |l|^2)
#define MPPI_SRHO(QW, QX, QY, QZ, RX, RY, RZ, EP)                                              \
    const float RX = fmaf(QW, QY, (QX) * (QZ)), RY = fmaf(-(QW), QX, (QY) * (QZ));             \
    float RZ, EP;                                                                              \
    {                                                                                          \
        const float n_ = fmaf(QZ, QZ, fmaf(QY, QY, fmaf(QX, QX, (QW) * (QW))));                \
        RZ = fmaf(0.5f, n_, -fmaf(QY, QY, (QX) * (QX)));                                       \
        EP = fmaf(-0.5f, n_, 0.5f);                                                            \
    }

template <int OBJ, int MATH, bool STORE_DU>
__global__ void __launch_bounds__(kScanThreads, 1) rollout_scan_kernel(const DevParams P, const StepArgs A)
{
    static_assert(OBJ == OBJ_GATE || OBJ == OBJ_GATE_PAPER, "time-parallel kernel: the two gate-progress objectives");
    extern __shared__ float4 smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, c = lane & (kScanC - 1), grp = lane >> 4;
    const int b = blockIdx.y, N = P.N, nthr = blockDim.x, nw = nthr >> 5;
    const int spb = nthr / kScanC;                     // samples per block
    const int kbase = blockIdx.x * spb;
    const int sidx = 2 * warp + grp;                   // this lane's sample within the block
    const uint32_t k = (uint32_t)(kbase + sidx);
    const bool valid = kbase + sidx < P.K;             // the last block of a controller may be ragged

    float4* s_unom = smem;
    float4* s_trk = smem + N;
    float* s_red = reinterpret_cast<float*>(s_trk + track_f4(P, OBJ));   // 64 floats
    float4* s_acc = reinterpret_cast<float4*>(s_red + 64);               // [16][N]
    float* s_cost = reinterpret_cast<float*>(s_acc + nw * N);            // [32]
    float* s_pair = s_cost + 32;                                         // 3 nb floats

    if (tid == 0) MPPI_STAMP(A, 0);
    const int L = (N + kScanC - 1) / kScanC;           // steps per chunk (<= kScanL)
    const int t0 = c * L;
    const int cnt = valid ? max(0, min(L, N - t0)) : 0;   // this lane's steps: t0 .. t0 + cnt - 1

    // ---- inputs.  The loads go out first and are parked in registers; the state-independent half of the noise
    //      (Philox, radius, angle: perturb_prepare) is drawn while they are in flight -- after an L2 flush they come
    //      from HBM -- and only then are they put into shared memory.  Under programmatic dependent launch
    //      (mppi_optimize's chain, StepArgs::pdl bit 0) the nominal is the previous kernel's output and is loaded after
    //      griddepcontrol.wait; gates, x0 and the draws do not depend on it.
    const bool pdl_wait = (A.pdl & 1) != 0;
    const float4* un_g = reinterpret_cast<const float4*>(A.u_nom) + (size_t)b * N;
    const int start = A.start[b];
    const State x0 = load_state(A.x0 + 13 * b);
    const int ng4 = 4 * P.G;                           // <= 4 MPPI_MAX_GATES = 256 <= 2 nthr
    float4 g_a = make_float4(0.f, 0.f, 0.f, 0.f), g_b = g_a, u_a = g_a;
    if (tid < ng4) g_a = P.gates[tid];
    if (tid + nthr < ng4) g_b = P.gates[tid + nthr];
    if (!pdl_wait && tid < N) u_a = un_g[tid];         // N <= 64 <= nthr
    float f[kScanL][4];
#pragma unroll
    for (int j = 0; j < kScanL; ++j)
        if (j < cnt) {
            const uint4 r = philox4x32_10(k, (uint32_t)(t0 + j), A.iter, (uint32_t)b, A.rk);
            perturb_prepare<MATH>(r.x, r.y, P.bm_k, f[j][0], f[j][1]);
            perturb_prepare<MATH>(r.z, r.w, P.bm_k, f[j][2], f[j][3]);
        }
    if (tid < ng4) s_trk[tid] = g_a;
    if (tid + nthr < ng4) s_trk[tid + nthr] = g_b;
    if (OBJ == OBJ_GATE_PAPER && tid <= N)             // previous-iteration "in front" flags (caller's; all ones without)
        reinterpret_cast<int*>(s_trk + ng4)[tid] = A.prev_front ? A.prev_front[(size_t)b * (N + 1) + tid] : 1;
    if (tid < 32) s_cost[tid] = __int_as_float(0x7f800000);      // samples this block does not have: cost +inf, weight 0
    if (pdl_wait) {
        asm volatile("griddepcontrol.wait;" ::: "memory");
        if (tid < N) u_a = un_g[tid];
    }
    if (tid < N) s_unom[tid] = u_a;
    __syncthreads();
    if (tid == 0) MPPI_STAMP(A, 1);

    // ---- eq.(3): the clamped thrusts of this lane's steps (second half of the pairs: the operations of
    //      sample_thrust), and what the dynamics need of them ----
    float4 T[kScanL];
    float ax[kScanL], ay[kScanL], az[kScanL], cm[kScanL];
#pragma unroll
    for (int j = 0; j < kScanL; ++j) {
        T[j] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (j < cnt) {
            const float4 un = s_unom[t0 + j];
            perturb_finish<MATH>(f[j][0], f[j][1], P.sigma, un.x, un.y, T[j].x, T[j].y);
            perturb_finish<MATH>(f[j][2], f[j][3], P.sigma, un.z, un.w, T[j].z, T[j].w);
            T[j].x = fminf(fmaxf(T[j].x, P.T_min), P.T_max); T[j].y = fminf(fmaxf(T[j].y, P.T_min), P.T_max);
            T[j].z = fminf(fmaxf(T[j].z, P.T_min), P.T_max); T[j].w = fminf(fmaxf(T[j].w, P.T_min), P.T_max);
            if (STORE_DU)
                A.du[((size_t)b * N + t0 + j) * P.K + k] = make_float4(T[j].x - un.x, T[j].y - un.y, T[j].z - un.z, T[j].w - un.w);
        }
        const float s01 = T[j].x + T[j].y, s23 = T[j].z + T[j].w;
        const float d10 = T[j].y - T[j].x, d23 = T[j].z - T[j].w;
        cm[j] = (s01 + s23) * P.inv_mass;              // S / m
        ax[j] = P.ltx * (s01 - s23);                   // tau_x / Jx
        ay[j] = P.lty * (d10 + d23);                   // tau_y / Jy
        az[j] = P.ltz * (d23 - d10);                   // tau_z / Jz
    }
    if (tid == 0) MPPI_STAMP(A, 2);

    // ---- omega_z: prefix sum of dt tau_z / Jz ----
    float oz_s;
    {
        float dz = 0.0f;
#pragma unroll
        for (int j = 0; j < kScanL; ++j)
            if (j < cnt) dz = fmaf(P.dt, az[j], dz);
        float inc = dz;
#pragma unroll
        for (int d = 1; d < kScanC; d <<= 1) {
            const float o = up16(inc, d);
            if (c >= d) inc += o;
        }
        const float prev = up16(inc, 1);               // exclusive
        oz_s = c ? x0.oz + prev : x0.oz;
    }

    // ---- omega_xy: the chunk's affine map w_end = H w_start + p (complex; H from the homogeneous run started at
    //      1, p from the particular run started at 0), then the scan over the chunks ----
    float ox_s, oy_s;
    {
        float hx = 1.0f, hy = 0.0f, px = 0.0f, py = 0.0f, oz = oz_s;
#pragma unroll
        for (int j = 0; j < kScanL; ++j)
            if (j < cnt) {
                const float z2 = fmaf(P.h2, az[j], oz), z4 = fmaf(P.dt, az[j], oz);
                omega_xy_step(P, hx, hy, 0.0f, 0.0f, oz, z2, z4);
                omega_xy_step(P, px, py, ax[j], ay[j], oz, z2, z4);
                oz = fmaf(P.h6, az[j], fmaf(P.h3, az[j], fmaf(P.h3, az[j], fmaf(P.h6, az[j], oz))));
            }
#pragma unroll
        for (int d = 1; d < kScanC; d <<= 1) {
            const float lhx = up16(hx, d), lhy = up16(hy, d), lpx = up16(px, d), lpy = up16(py, d);
            if (c >= d) {                              // (H, p) o (lH, lp): the left operand acts first
                const float nhx = fmaf(hx, lhx, -hy * lhy), nhy = fmaf(hx, lhy, hy * lhx);
                px = fmaf(hx, lpx, fmaf(-hy, lpy, px));
                py = fmaf(hx, lpy, fmaf(hy, lpx, py));
                hx = nhx; hy = nhy;
            }
        }
        const float ex = fmaf(hx, x0.ox, fmaf(-hy, x0.oy, px)), ey = fmaf(hx, x0.oy, fmaf(hy, x0.ox, py));   // omega_xy after chunk c
        const float sx = up16(ex, 1), sy = up16(ey, 1);
        ox_s = c ? sx : x0.ox;
        oy_s = c ? sy : x0.oy;
    }
    if (tid == 0) MPPI_STAMP(A, 4);

    // ---- attitude and translation of the chunk in its own frame: the RK4 of rk4_step from (omega_s, l = identity);
    //      lane 0 starts from q0 itself (its frame is the world frame), so an x0 whose quaternion is not normalised
    //      is treated as rk4_step treats it ----
    float lw = c ? 1.0f : x0.qw, lx = c ? 0.0f : x0.qx, ly = c ? 0.0f : x0.qy, lz = c ? 0.0f : x0.qz;
    float Vx = 0.0f, Vy = 0.0f, Vz = 0.0f, Ve = 0.0f;       // chunk-frame velocity gained (rotating part, world-z part)
    float Px[kScanL], Py[kScanL], Pz[kScanL], Pe[kScanL];   // chunk-frame position gained after step j
    float w2 = 0.0f;                                        // sum |omega_{t+1}|^2
    {
        float ox = ox_s, oy = oy_s, oz = oz_s;
        float prx = 0.0f, pry = 0.0f, prz = 0.0f, pre = 0.0f;
        const float gh = P.dt * P.g, ghh = P.hh2 * P.g;
#pragma unroll
        for (int j = 0; j < kScanL; ++j) {
            if (j < cnt) {
                const float kp = cm[j] * P.hh3, kv = cm[j] * P.h3;
                const float a_x = ax[j], a_y = ay[j], a_z = az[j];
                // stage 1
                float kox = fmaf(P.gyx, oy * oz, a_x), koy = fmaf(P.gyy, oz * ox, a_y);
                float gw, gx, gy, gz;
                MPPI_SG(lw, lx, ly, lz, ox, oy, oz, gw, gx, gy, gz)
                MPPI_SRHO(lw, lx, ly, lz, r1x, r1y, r1z, e1)
                float nox = fmaf(P.h6, kox, ox), noy = fmaf(P.h6, koy, oy), noz = fmaf(P.h6, a_z, oz);
                float nw = fmaf(P.h12, gw, lw), nx = fmaf(P.h12, gx, lx), ny = fmaf(P.h12, gy, ly), nz = fmaf(P.h12, gz, lz);
                float sx = fmaf(P.h2, kox, ox), sy = fmaf(P.h2, koy, oy), sz = fmaf(P.h2, a_z, oz);
                float qw = fmaf(P.h4, gw, lw), qx = fmaf(P.h4, gx, lx), qy = fmaf(P.h4, gy, ly), qz = fmaf(P.h4, gz, lz);
                // stage 2
                kox = fmaf(P.gyx, sy * sz, a_x); koy = fmaf(P.gyy, sz * sx, a_y);
                MPPI_SG(qw, qx, qy, qz, sx, sy, sz, gw, gx, gy, gz)
                MPPI_SRHO(qw, qx, qy, qz, r2x, r2y, r2z, e2)
                nox = fmaf(P.h3, kox, nox); noy = fmaf(P.h3, koy, noy); noz = fmaf(P.h3, a_z, noz);
                nw = fmaf(P.h6, gw, nw); nx = fmaf(P.h6, gx, nx); ny = fmaf(P.h6, gy, ny); nz = fmaf(P.h6, gz, nz);
                sx = fmaf(P.h2, kox, ox); sy = fmaf(P.h2, koy, oy);
                qw = fmaf(P.h4, gw, lw); qx = fmaf(P.h4, gx, lx); qy = fmaf(P.h4, gy, ly); qz = fmaf(P.h4, gz, lz);
                // stage 3
                kox = fmaf(P.gyx, sy * sz, a_x); koy = fmaf(P.gyy, sz * sx, a_y);
                MPPI_SG(qw, qx, qy, qz, sx, sy, sz, gw, gx, gy, gz)
                MPPI_SRHO(qw, qx, qy, qz, r3x, r3y, r3z, e3)
                nox = fmaf(P.h3, kox, nox); noy = fmaf(P.h3, koy, noy); noz = fmaf(P.h3, a_z, noz);
                nw = fmaf(P.h6, gw, nw); nx = fmaf(P.h6, gx, nx); ny = fmaf(P.h6, gy, ny); nz = fmaf(P.h6, gz, nz);
                sx = fmaf(P.dt, kox, ox); sy = fmaf(P.dt, koy, oy); sz = fmaf(P.dt, a_z, oz);
                qw = fmaf(P.h2, gw, lw); qx = fmaf(P.h2, gx, lx); qy = fmaf(P.h2, gy, ly); qz = fmaf(P.h2, gz, lz);
                // stage 4
                kox = fmaf(P.gyx, sy * sz, a_x); koy = fmaf(P.gyy, sz * sx, a_y);
                MPPI_SG(qw, qx, qy, qz, sx, sy, sz, gw, gx, gy, gz)
                MPPI_SRHO(qw, qx, qy, qz, r4x, r4y, r4z, e4)
                ox = fmaf(P.h6, kox, nox); oy = fmaf(P.h6, koy, noy); oz = fmaf(P.h6, a_z, noz);
                nw = fmaf(P.h12, gw, nw); nx = fmaf(P.h12, gx, nx); ny = fmaf(P.h12, gy, ny); nz = fmaf(P.h12, gz, nz);
                // translation in the chunk frame: A = sum of stages 1..3, B = 1, 2, 2, 1 weights
                const float mx = r2x + r3x, my = r2y + r3y, mz = r2z + r3z, me = e2 + e3;
                const float Ax = r1x + mx, Ay = r1y + my, Az = r1z + mz, Ae = e1 + me;
                prx = fmaf(kp, Ax, fmaf(P.dt, Vx, prx));
                pry = fmaf(kp, Ay, fmaf(P.dt, Vy, pry));
                prz = fmaf(kp, Az, fmaf(P.dt, Vz, prz));
                pre = fmaf(kp, Ae, fmaf(P.dt, Ve, pre)) - ghh;
                Vx = fmaf(kv, (Ax + mx) + r4x, Vx);
                Vy = fmaf(kv, (Ay + my) + r4y, Vy);
                Vz = fmaf(kv, (Az + mz) + r4z, Vz);
                Ve = fmaf(kv, (Ae + me) + e4, Ve) - gh;
                const float inv = MATH == 0 ? rsqrtf(fmaf(nz, nz, fmaf(ny, ny, fmaf(nx, nx, nw * nw))))
                                            : mufu_rsq(fmaf(nz, nz, fmaf(ny, ny, fmaf(nx, nx, nw * nw))));
                lw = nw * inv; lx = nx * inv; ly = ny * inv; lz = nz * inv;
                w2 = fmaf(oz, oz, fmaf(oy, oy, fmaf(ox, ox, w2)));
            }
            Px[j] = prx; Py[j] = pry; Pz[j] = prz; Pe[j] = pre;
        }
    }
    if (tid == 0) MPPI_STAMP(A, 5);

    // ---- chunk start attitudes: inclusive scan of the chunk quaternions (lane 0's carries q0), shifted by one ----
    float sw, sx_, sy_, sz_;                            // q_s: attitude at the start of this chunk (identity for lane 0)
    {
        float aw = lw, ax_ = lx, ay_ = ly, az_ = lz;
#pragma unroll
        for (int d = 1; d < kScanC; d <<= 1) {
            const float bw = up16(aw, d), bx = up16(ax_, d), by = up16(ay_, d), bz = up16(az_, d);
            if (c >= d) {                              // left (x) mine
                const float nw = fmaf(-bz, az_, fmaf(-by, ay_, fmaf(-bx, ax_, bw * aw)));
                const float nx = fmaf(-bz, ay_, fmaf(by, az_, fmaf(bx, aw, bw * ax_)));
                const float ny = fmaf(bz, ax_, fmaf(by, aw, fmaf(-bx, az_, bw * ay_)));
                const float nz = fmaf(bz, aw, fmaf(-by, ax_, fmaf(bx, ay_, bw * az_)));
                aw = nw; ax_ = nx; ay_ = ny; az_ = nz;
            }
        }
        const float inv = rsqrtf(fmaf(az_, az_, fmaf(ay_, ay_, fmaf(ax_, ax_, aw * aw))));
        aw *= inv; ax_ *= inv; ay_ *= inv; az_ *= inv;
        const float pw = up16(aw, 1), pxq = up16(ax_, 1), pyq = up16(ay_, 1), pzq = up16(az_, 1);
        sw = c ? pw : 1.0f; sx_ = c ? pxq : 0.0f; sy_ = c ? pyq : 0.0f; sz_ = c ? pzq : 0.0f;
    }
    // R(q_s)
    const float R00 = 1.0f - 2.0f * fmaf(sy_, sy_, sz_ * sz_), R01 = 2.0f * fmaf(sx_, sy_, -sw * sz_), R02 = 2.0f * fmaf(sx_, sz_, sw * sy_);
    const float R10 = 2.0f * fmaf(sx_, sy_, sw * sz_), R11 = 1.0f - 2.0f * fmaf(sx_, sx_, sz_ * sz_), R12 = 2.0f * fmaf(sy_, sz_, -sw * sx_);
    const float R20 = 2.0f * fmaf(sx_, sz_, -sw * sy_), R21 = 2.0f * fmaf(sy_, sz_, sw * sx_), R22 = 1.0f - 2.0f * fmaf(sx_, sx_, sy_ * sy_);

    // ---- velocities, then positions: two prefix sums over the chunks ----
    float vsx, vsy, vsz, psx, psy, psz;                 // world velocity / position at the start of this chunk
    {
        float dx = fmaf(R02, Vz, fmaf(R01, Vy, R00 * Vx)), dy = fmaf(R12, Vz, fmaf(R11, Vy, R10 * Vx)),
              dz = fmaf(R22, Vz, fmaf(R21, Vy, R20 * Vx)) + Ve;
#pragma unroll
        for (int d = 1; d < kScanC; d <<= 1) {
            const float ux = up16(dx, d), uy = up16(dy, d), uz = up16(dz, d);
            if (c >= d) { dx += ux; dy += uy; dz += uz; }
        }
        const float ux = up16(dx, 1), uy = up16(dy, 1), uz = up16(dz, 1);
        vsx = c ? x0.vx + ux : x0.vx; vsy = c ? x0.vy + uy : x0.vy; vsz = c ? x0.vz + uz : x0.vz;
        const int last = cnt > 0 ? cnt - 1 : 0;
        float ex = 0.0f, ey = 0.0f, ez = 0.0f, ee = 0.0f;          // chunk-frame position gained over the whole chunk
#pragma unroll
        for (int j = 0; j < kScanL; ++j)
            if (j == last) { ex = Px[j]; ey = Py[j]; ez = Pz[j]; ee = Pe[j]; }
        const float span = (float)cnt * P.dt;
        dx = fmaf(span, vsx, fmaf(R02, ez, fmaf(R01, ey, R00 * ex)));
        dy = fmaf(span, vsy, fmaf(R12, ez, fmaf(R11, ey, R10 * ex)));
        dz = fmaf(span, vsz, fmaf(R22, ez, fmaf(R21, ey, R20 * ex)) + ee);
#pragma unroll
        for (int d = 1; d < kScanC; d <<= 1) {
            const float wx = up16(dx, d), wy = up16(dy, d), wz = up16(dz, d);
            if (c >= d) { dx += wx; dy += wy; dz += wz; }
        }
        const float wx = up16(dx, 1), wy = up16(dy, 1), wz = up16(dz, 1);
        psx = c ? x0.px + wx : x0.px; psy = c ? x0.py + wy : x0.py; psz = c ? x0.pz + wz : x0.pz;
    }
    // world positions after each of this lane's steps (x_{t+1}, t = t0 + j), in place
#pragma unroll
    for (int j = 0; j < kScanL; ++j) {
        const float tt = (float)(j + 1) * P.dt;
        const float ex = Px[j], ey = Py[j], ez = Pz[j];
        Px[j] = fmaf(tt, vsx, psx) + fmaf(R02, ez, fmaf(R01, ey, R00 * ex));
        Py[j] = fmaf(tt, vsy, psy) + fmaf(R12, ez, fmaf(R11, ey, R10 * ex));
        Pz[j] = fmaf(tt, vsz, psz) + (fmaf(R22, ez, fmaf(R21, ey, R20 * ex)) + Pe[j]);
    }
    // The position before this lane's first step is the previous lane's last one -- taken from there, bit for bit,
    // so that the lanes score one and the same sequence of positions (crossing tests and distances at a chunk
    // boundary are then the same numbers on both sides of it).
    {
        const int last = cnt > 0 ? cnt - 1 : 0;
        float ex = 0.0f, ey = 0.0f, ez = 0.0f;
#pragma unroll
        for (int j = 0; j < kScanL; ++j)
            if (j == last) { ex = Px[j]; ey = Py[j]; ez = Pz[j]; }
        const float ux = up16(ex, 1), uy = up16(ey, 1), uz = up16(ez, 1);
        psx = c ? ux : x0.px; psy = c ? uy : x0.py; psz = c ? uz : x0.pz;
    }
    if (tid == 0) MPPI_STAMP(A, 6);

    // ---- objective ----
    float J;
    {
        // GateCost / GatePaperCost (mppi_cost.cuh) chunk by chunk.  Across a chunk boundary the state of the machine
        // is the target index alone (s_prev and the segment's first distance are functions of the boundary position;
        // the paper's form also looks at the horizon's start gate, a constant), and a chunk's progress
        // |p_end - c| - |p_start - c| is its own telescoped segment.
        const float4* s_gates = s_trk;
        const int* s_front = reinterpret_cast<const int*>(s_trk + 4 * P.G);      // OBJ_GATE_PAPER only
        const int gate0 = wrap_index(start, P.G);
        int g_in = gate0, g_out = g_in, lo = 0;
        bool need = true;
        float Jc = 0.0f;
        const unsigned gmask = 0xffffu << (lane & 16);
        for (;;) {
            if (need && OBJ == OBJ_GATE_PAPER) {
                // eq.(6),(7) with squared distances, the near-gate term on the pre-step state and the temporal
                // check of Fig. 2 [R-23]..[R-25], [R-40]: GatePaperCost::step, operation for operation
                int gate = g_in;
                float4 cg = s_gates[4 * gate], ng = s_gates[4 * gate + 1];
                float ppx = psx, ppy = psy, ppz = psz;
                float rx0 = ppx - cg.x, ry0 = ppy - cg.y, rz0 = ppz - cg.z;
                float d2_0 = fmaf(rz0, rz0, fmaf(ry0, ry0, rx0 * rx0)), d2_prev = d2_0;
                float s_prev = fmaf(ng.z, rz0, fmaf(ng.y, ry0, ng.x * rx0));
                float acc = 0.0f;
#pragma unroll
                for (int j = 0; j < kScanL; ++j)
                    if (j < cnt) {
                        const float px = Px[j], py = Py[j], pz = Pz[j];
                        float dn2 = d2_prev;
                        if (P.near_mode == 1 && gate != gate0) {
                            const float4 c0 = s_gates[4 * gate0];
                            const float ux = ppx - c0.x, uy = ppy - c0.y, uz = ppz - c0.z;
                            dn2 = fmaf(uz, uz, fmaf(uy, uy, ux * ux));
                        }
                        if (dn2 < P.r_near2) acc = fmaf(P.q_near, dn2, acc);
                        const float fx = px - cg.x, fy = py - cg.y, fz = pz - cg.z;
                        const float d2 = fmaf(fz, fz, fmaf(fy, fy, fx * fx));
                        const float s = fmaf(ng.z, fz, fmaf(ng.y, fy, ng.x * fx));
                        bool switched = false;
                        if (s_prev < 0.0f && s >= 0.0f) {                 // front -> back through the plane
                            const float4 hg = s_gates[4 * gate + 2], vg = s_gates[4 * gate + 3];
                            const float alpha = s_prev / (s_prev - s);
                            const float rx = ppx - cg.x, ry = ppy - cg.y, rz = ppz - cg.z;
                            const float hx = fmaf(alpha, fx - rx, rx), hy = fmaf(alpha, fy - ry, ry), hz = fmaf(alpha, fz - rz, rz);
                            const float y = fmaf(hg.z, hz, fmaf(hg.y, hy, hg.x * hx));
                            const float z = fmaf(vg.z, hz, fmaf(vg.y, hy, vg.x * hx));
                            if (fabsf(y) <= cg.w && fabsf(z) <= ng.w) {
                                if (gate != gate0 || s_front[t0 + j + 1] != 0) {      // temporally consistent pass
                                    acc += (d2 - d2_0) - P.bonus;                     // close the segment
                                    gate = (gate + 1 == P.G) ? 0 : gate + 1;
                                    cg = s_gates[4 * gate]; ng = s_gates[4 * gate + 1];
                                    const float qx = px - cg.x, qy = py - cg.y, qz = pz - cg.z;
                                    d2_0 = fmaf(qz, qz, fmaf(qy, qy, qx * qx)); d2_prev = d2_0;
                                    s_prev = fmaf(ng.z, qz, fmaf(ng.y, qy, ng.x * qx));
                                    switched = true;
                                }
                            } else {
                                acc += P.miss;                                        // miss: target unchanged
                            }
                        }
                        if (!switched) { s_prev = s; d2_prev = d2; }
                        ppx = px; ppy = py; ppz = pz;
                    }
                Jc = acc + (d2_prev - d2_0);
                g_out = gate;
            }
            if (need && OBJ == OBJ_GATE) {
                int gate = g_in;
                float4 cg = s_gates[4 * gate], ng = s_gates[4 * gate + 1], hg = s_gates[4 * gate + 2];
                float d0 = GateCost::norm3<MATH>(psx - cg.x, psy - cg.y, psz - cg.z);
                float s_prev = GateCost::plane(ng, hg.w, psx, psy, psz);
                float ppx = psx, ppy = psy, ppz = psz;
                float acc = 0.0f;
#pragma unroll
                for (int j = 0; j < kScanL; ++j)
                    if (j < cnt) {
                        const float px = Px[j], py = Py[j], pz = Pz[j];
                        const float s = GateCost::plane(ng, hg.w, px, py, pz);
                        if (s_prev < 0.0f && s >= 0.0f) {                 // front -> back through the plane
                            const float4 vg = s_gates[4 * gate + 3];
                            const float fx = px - cg.x, fy = py - cg.y, fz = pz - cg.z;
                            const float alpha = s_prev / (s_prev - s);
                            const float rx = ppx - cg.x, ry = ppy - cg.y, rz = ppz - cg.z;
                            const float hx = fmaf(alpha, fx - rx, rx), hy = fmaf(alpha, fy - ry, ry), hz = fmaf(alpha, fz - rz, rz);
                            const float y = fmaf(hg.z, hz, fmaf(hg.y, hy, hg.x * hx));
                            const float z = fmaf(vg.z, hz, fmaf(vg.y, hy, vg.x * hx));
                            if (fabsf(y) <= cg.w && fabsf(z) <= ng.w) {   // inside the opening: pass + switch
                                acc += (GateCost::norm3<MATH>(fx, fy, fz) - d0) - P.bonus;
                                gate = (gate + 1 == P.G) ? 0 : gate + 1;
                                cg = s_gates[4 * gate]; ng = s_gates[4 * gate + 1]; hg = s_gates[4 * gate + 2];
                                d0 = GateCost::norm3<MATH>(px - cg.x, py - cg.y, pz - cg.z);
                                s_prev = GateCost::plane(ng, hg.w, px, py, pz);
                            } else {                                      // miss: target unchanged
                                acc += P.miss;
                                s_prev = s;
                            }
                        } else {
                            s_prev = s;
                        }
                        ppx = px; ppy = py; ppz = pz;
                    }
                Jc = acc + (GateCost::norm3<MATH>(ppx - cg.x, ppy - cg.y, ppz - cg.z) - d0);
                g_out = gate;
            }
            // first lane, in horizon order, of the still unconfirmed ones whose chunk switches the target
            const unsigned ch = __ballot_sync(kFull, g_out != g_in && c >= lo) & gmask;
            const bool done = ch == 0u;
            const int first = done ? lane : __ffs(ch) - 1;
            const int ng_ = __shfl_sync(kFull, g_out, first);
            need = !done && lane > first;
            if (need) g_in = ng_;
            lo = done ? kScanC : (first & (kScanC - 1)) + 1;
            if (!__any_sync(kFull, !done)) break;
        }
        J = fmaf(P.w_omega, w2, Jc);
    }
    // sum over the sample's 16 lanes (fixed butterfly: deterministic)
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) J += __shfl_xor_sync(kFull, J, o);
    J = sanitize_cost(J);
    if (c == 0 && valid) s_cost[sidx] = J;
    // the rollouts of this block are through: a dependent launch (the next iteration of mppi_optimize's chain) may
    // be brought up; its blocks draw their normals and wait for this grid before they read the nominal
    if (A.pdl & 2) asm volatile("griddepcontrol.launch_dependents;");
    __syncthreads();
    if (tid == 0) MPPI_STAMP(A, 7);

    // ---- block partial of the fused update (eq.(4),(5)).  With 14-16 warps on the SM every instruction of this
    //      tail costs ~4 cycles of wall time, so it is kept short: every warp forms the block minimum and the 32 weights
    //      on its own (one CREDUX), only the warps that hold a sample with a non-zero weight -- every warp knows which
    //      those are -- weigh their perturbations and take part in the sum over the warps (in the near-arg-min regime of
    //      the paper's lambda that is one or two warps), and Z is formed by warp 0 beside the others' stores ----
    const float Jl = s_cost[lane];
    const bool have = lane < spb && kbase + lane < P.K;
    if (warp == 0 && have) A.cost[(size_t)b * P.K + kbase + lane] = Jl;
    const float m = warp_min(Jl);
    const float el = have ? exp_weight<MATH>((m - Jl) * P.inv_lambda) : 0.0f;
    const unsigned cmask = __ballot_sync(kFull, el != 0.0f);      // samples of the block that carry weight
    if ((cmask >> (2 * warp)) & 3u) {
        const float e = __shfl_sync(kFull, el, sidx);
#pragma unroll
        for (int j = 0; j < kScanL; ++j) {
            float4 d = make_float4(0.f, 0.f, 0.f, 0.f);
            if (j < cnt) {
                const float4 un = s_unom[t0 + j];
                d = make_float4(e * (T[j].x - un.x), e * (T[j].y - un.y), e * (T[j].z - un.z), e * (T[j].w - un.w));
            }
            d = add4(d, shfl_xor4(d, 16));
            if (grp == 0 && j < cnt) s_acc[warp * N + t0 + j] = d;
        }
    }
    float Zb = 0.0f;
    if (warp == 0) Zb = warp_sum(el);
    __syncthreads();
    if (tid == 0) MPPI_STAMP(A, 3);
    float* part = A.partials + ((size_t)b * P.blocks_per_ctrl + blockIdx.x) * P.part_stride;
    for (int j = tid; j < 4 * N; j += nthr) {
        float s = 0.0f;
        for (unsigned mm = cmask; mm; ) {              // contributing warps in ascending order: deterministic
            const int w = (__ffs(mm) - 1) >> 1;
            mm &= ~(3u << (2 * w));
            s += reinterpret_cast<const float*>(s_acc)[w * 4 * N + j];
        }
        part[j] = s;
    }
    if (tid == 0) write_partial_header(P, A, b, blockIdx.x, m, Zb);
    publish_and_combine<MATH, 4>(P, A, b, P.blocks_per_ctrl, s_unom, s_red, s_pair, reinterpret_cast<float*>(s_acc));
    if (tid == 0) MPPI_STAMP(A, 12);
}

#undef MPPI_SG
#undef MPPI_SRHO

}  // namespace mppi
