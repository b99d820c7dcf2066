// mppi_kernels.cu -- the sm_100a kernels of the MPPI hot path.
//
//   rollout_kernel<OBJ, MATH, STORE_DU, FUSED>   SURVEY.md 8(a) steps 1-4 (+5-7 when FUSED), one sample
//                                                per thread, noise drawn in the horizon loop (throughput)
//   rollout_lat_kernel<OBJ, MATH, STORE_DU>      the same iteration for a lone controller (latency):
//                                                all warps draw the noise first, few warps roll out
//   reduce_kernel                                steps 5-7 of the TWO_PASS pipeline
//   sim_kernel                                   step 8 (closed-loop glue)
//
// No tensor cores: nothing here is a contraction.
#include <cstring>
#include "mppi_internal.h"
#include "mppi_rollout.cuh"
#include "mppi_packed.cuh"
#include "mppi_pipe.cuh"
#include "mppi_rate.cuh"
#include "mppi_pipe_rate.cuh"

namespace mppi {

constexpr int kLatChunk = 5;       // steps per hand-over of the contouring split of rollout_lat_kernel
__host__ __device__ inline int lat_chunks(int N) { return (N + kLatChunk - 1) / kLatChunk; }

// float4 units of the register-pair rows of the contouring candidates (nearest_rot4, packed kernel); 0 = not used
__host__ __device__ inline int contour_pair_f4(const DevParams& P)
{
    return (P.window == 16 && P.P <= 1024) ? 2 * (P.P + 2 * P.window + 14) : 0;
}

// Shared-memory carve-up of rollout_kernel (units: float4).
//   [0, N)                         nominal thrusts u_nom[b]
//   [N, N + trk)                   track data of the objective
//   then 16 float4                 reduction scratch (64 floats)
//   FUSED: nwarps * N float4       per-warp weighted-noise accumulators
//   FUSED: ceil(3 nblk / 4) float4 (min, Z) pairs / rescale factors / index list of the last-block combine
size_t rollout_smem_bytes(const DevParams& P, const LaunchCfg& c)
{
    size_t f4 = (size_t)P.N + track_f4(P, c.objective) + 16;
    if (c.scan) return scan_smem_bytes(P, c);
    if (c.pipe) return (f4 + (c.rate ? pipe_rate_extra_f4(P.N, P.blocks_per_ctrl, c.objective == OBJ_CONTOUR_PAPER, P.pipe_d, P.pipe_df) : pipe_extra_f4(P.N, P.blocks_per_ctrl))) * sizeof(float4);
    if (c.lat_consumers > 0) {
        f4 += (size_t)P.N * (32 * c.lat_consumers + 1) + 32 + (3 * P.blocks_per_ctrl + 3) / 4;
        if (c.objective == OBJ_CONTOUR && c.lat_split)   // rollout warps -> search warps: positions [N][32 C], costs [32 C], mbarriers
            f4 += (size_t)P.N * 32 * c.lat_consumers + 8 * c.lat_consumers + (c.lat_consumers * lat_chunks(P.N) + 1) / 2 + contour_pair_f4(P);
        return f4 * sizeof(float4);
    }
    if (c.fused) f4 += (size_t)(c.block_threads / 32) * P.N + (3 * P.blocks_per_ctrl + 3) / 4;
    if (c.packed && c.objective == OBJ_CONTOUR) f4 += contour_pair_f4(P);     // candidate pairs of nearest_rot4
    if (c.objective == OBJ_CONTOUR_PAPER)      // fifth column: its nominal + one accumulator row per warp
        f4 += ((size_t)(c.block_threads / 32 + 1) * P.N + 3) / 4;
    return f4 * sizeof(float4);
}

// ---------------------------------------------------------------------------------------------
// packed throughput variant: two samples per thread in fp32x2 registers (mppi_packed.cuh).
// grid = (K / (2 blockDim.x), B); thread j of the grid row owns samples 2j and 2j+1.
// ---------------------------------------------------------------------------------------------
// ---------------------------------------------------------------------------------------------
// Windowed nearest-vertex search of objective 2 for the packed kernel, FOUR candidates per round in packed fp32x2
// arithmetic.  configs[3] x 64 was bound by issue slots (75 % busy) AND by the shared-memory pipe (0.72 wavefronts
// per SM-cycle), two thirds of both being this search (profiles/README_r02c.md).  The candidates of the padded copy
// (ContourCost::nearest_ext) are laid out a second time so that register PAIRS come straight out of 128-bit loads:
//   xy2[j] = (x_j, x_{j+1}, y_j, y_{j+1})      z4[j] = (z_j, z_{j+1}, z_{j+2}, z_{j+3})
// Per four candidates: 3 LDS.128 (12 bytes per candidate instead of 16), 6 FADD2 + 2 FMUL2 + 4 FFMA2 (instead of 24
// scalar operations), then the four compare-and-selects in scan order.  Same rotation as nearest_rot (each lane starts
// at the entry congruent to its lane number mod 8: conflict-free 128-bit loads), same distances (dx dx, then + dy dy,
// then + dz dz), same strict comparison in the same order: the same minimiser, bit for bit.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ int nearest_rot4(const DevParams& P, const float4* __restrict__ xy2, const float4* __restrict__ z4,
                                            const int centre, const float px, const float py, const float pz)
{
    constexpr int W = 16, n = 2 * W + 1, PAD = ContourCost::kExtPad;
    const int ws = centre + PAD;                             // window start in the padded copy
    const int r = (ws - (int)(threadIdx.x & 7)) & 7;
    const int jb = ws - r;
    const float2 PX = bc2(px), PY = bc2(py), PZ = bc2(pz);
    const float inf = __int_as_float(0x7f800000);
    float best = inf;
    int ob = W + r;
#pragma unroll
    for (int o = 0; o < n + PAD; o += 4) {
        const float4 a0 = xy2[jb + o], a1 = xy2[jb + o + 2], zz = z4[jb + o];
        const float2 dx0 = sub2(PX, make_float2(a0.x, a0.y)), dy0 = sub2(PY, make_float2(a0.z, a0.w)), dz0 = sub2(PZ, make_float2(zz.x, zz.y));
        const float2 dx1 = sub2(PX, make_float2(a1.x, a1.y)), dy1 = sub2(PY, make_float2(a1.z, a1.w)), dz1 = sub2(PZ, make_float2(zz.z, zz.w));
        const float2 e0 = fma2(dz0, dz0, fma2(dy0, dy0, mul2(dx0, dx0)));
        const float2 e1 = fma2(dz1, dz1, fma2(dy1, dy1, mul2(dx1, dx1)));
        float d[4] = {e0.x, e0.y, e1.x, e1.y};
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int oo = o + q;
            if (oo < PAD) d[q] = oo >= r ? d[q] : inf;
            if (oo >= n) d[q] = oo <= r + 2 * W ? d[q] : inf;
            if (d[q] < best) { best = d[q]; ob = oo; }
        }
    }
    int i = centre + (ob - r) - W;
    if (P.closed) { if (i < 0) i += P.P; else if (i >= P.P) i -= P.P; }
    return i;
}

template <int OBJ, int MATH, bool SYMZ>
__device__ __forceinline__ void rollout_cost2(const DevParams& P, const StepArgs& A, const float4* s_unom,
                                              const float4* s_trk, State2 x, int start, int contour_i0,
                                              uint32_t k0, uint32_t b, float4* du_out, float& Ja, float& Jb,
                                              const float4* s_xy2 = nullptr, const float4* s_z4 = nullptr)
{
    const int N = P.N;
    Ja = 0.0f; Jb = 0.0f;
    GateCost ga, gb;
    GatePaperCost pa, pb;
    ContourCost ca, cb;
    const int* s_front = reinterpret_cast<const int*>(s_trk + 4 * P.G);      // OBJ_GATE_PAPER only
    if (OBJ == OBJ_GATE) { ga.init<MATH>(P, s_trk, start, lane_state<0>(x)); gb = ga; }
    if (OBJ == OBJ_GATE_PAPER) { pa.init(P, s_trk, start, lane_state<0>(x)); pb = pa; }
    if (OBJ == OBJ_CONTOUR) { ca.init(P, s_trk, contour_i0, lane_state<0>(x)); cb = ca; }
    for (int t = 0; t < N; ++t) {
        const float4 un = s_unom[t];
        const float4 Ta = sample_thrust<MATH>(P, A.rk, k0, (uint32_t)t, A.iter, b, un);
        const float4 Tb = sample_thrust<MATH>(P, A.rk, k0 + 1u, (uint32_t)t, A.iter, b, un);
        if (du_out) {
            du_out[(size_t)t * P.K] = make_float4(Ta.x - un.x, Ta.y - un.y, Ta.z - un.z, Ta.w - un.w);
            du_out[(size_t)t * P.K + 1] = make_float4(Tb.x - un.x, Tb.y - un.y, Tb.z - un.z, Tb.w - un.w);
        }
        if (OBJ == OBJ_TRACK) {
            Ja += track_stage(P, s_trk + 4 * t, lane_state<0>(x), Ta);
            Jb += track_stage(P, s_trk + 4 * t, lane_state<1>(x), Tb);
        }
        rk4_step2<SYMZ>(P, x, Ta, Tb);
        if (OBJ == OBJ_GATE) {
            ga.step<MATH>(P, s_trk, lane_state<0>(x));
            gb.step<MATH>(P, s_trk, lane_state<1>(x));
        }
        if (OBJ == OBJ_GATE_PAPER) {
            pa.step(P, s_trk, s_front, lane_state<0>(x), t);
            pb.step(P, s_trk, s_front, lane_state<1>(x), t);
        }
        if (OBJ == OBJ_CONTOUR) {
            if (s_xy2) {                                                  // four candidates per round (nearest_rot4)
                const State xa = lane_state<0>(x), xb = lane_state<1>(x);
                ca.idx = nearest_rot4(P, s_xy2, s_z4, ca.idx, xa.px, xa.py, xa.pz);
                cb.idx = nearest_rot4(P, s_xy2, s_z4, cb.idx, xb.px, xb.py, xb.pz);
                Ja += ca.step_found(P, s_trk, xa.px, xa.py, xa.pz, xa.ox * xa.ox + xa.oy * xa.oy + xa.oz * xa.oz);
                Jb += cb.step_found(P, s_trk, xb.px, xb.py, xb.pz, xb.ox * xb.ox + xb.oy * xb.oy + xb.oz * xb.oz);
            } else {
                Ja += ca.template step<true>(P, s_trk, lane_state<0>(x));     // conflict-free scan (nearest_rot)
                Jb += cb.template step<true>(P, s_trk, lane_state<1>(x));
            }
        }
    }
    if (OBJ == OBJ_GATE) {
        Ja = ga.finish<MATH>(P, s_trk, lane_state<0>(x));
        Jb = gb.finish<MATH>(P, s_trk, lane_state<1>(x));
    }
    if (OBJ == OBJ_GATE_PAPER) { Ja = pa.finish(P); Jb = pb.finish(P); }
    if (OBJ == OBJ_TRACK) {
        Ja += track_state_term(P, s_trk + 4 * N, lane_state<0>(x));
        Jb += track_state_term(P, s_trk + 4 * N, lane_state<1>(x));
    }
}

#ifndef MPPI_PK_THREADS
#define MPPI_PK_THREADS 128     // max block size of the packed kernel
#define MPPI_PK_MINB 4          // resident blocks per SM the register budget is sized for
#endif
template <int OBJ, int MATH, bool STORE_DU, bool FUSED>
__global__ void __launch_bounds__(MPPI_PK_THREADS, MPPI_PK_MINB) rollout2_kernel(const DevParams P, const StepArgs A)
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

    const int start = A.start[b];
    stage_inputs<OBJ>(P, A, b, start, s_unom, s_trk);
    __syncthreads();

    // objective 2: the candidates once more as register-pair rows for nearest_rot4 (after the combine scratch)
    float4* s_xy2 = nullptr; float4* s_z4 = nullptr;
    if (OBJ == OBJ_CONTOUR && contour_pair_f4(P) > 0) {
        const int L = P.P + 2 * P.window + 14;
        const float4* ext = s_trk + 2 * P.P;
        s_xy2 = FUSED ? reinterpret_cast<float4*>(s_pair) + (3 * P.blocks_per_ctrl + 3) / 4 : s_acc;      // (two-pass: no combine scratch)
        s_z4 = s_xy2 + L;
        for (int j = tid; j < L; j += blockDim.x) {
            const float4 e0 = ext[j], e1 = ext[min(j + 1, L - 1)], e2 = ext[min(j + 2, L - 1)], e3 = ext[min(j + 3, L - 1)];
            const float far = 1e30f;                                   // beyond the copy: never the minimum
            s_xy2[j] = make_float4(e0.x, j + 1 < L ? e1.x : far, e0.y, j + 1 < L ? e1.y : far);
            s_z4[j] = make_float4(e0.z, j + 1 < L ? e1.z : far, j + 2 < L ? e2.z : far, j + 3 < L ? e3.z : far);
        }
    }
    const State x0 = load_state(A.x0 + 13 * b);
    const int i0 = OBJ == OBJ_CONTOUR ? contour_start_index(P, s_trk, start, x0, s_red) : 0;
    if (OBJ == OBJ_CONTOUR) __syncthreads();
    float Ja, Jb;
    const bool stored = FUSED ? keeps_du<STORE_DU>(A, b) : STORE_DU;
    float4* const du_out = stored ? A.du + (size_t)b * N * P.K + k0 : nullptr;
    if (OBJ != OBJ_CONTOUR && P.gyz == 0.0f)       // (the contouring search is bound by shared memory) Jx == Jy: the yaw-rate derivative is constant over the step (rk4_step2<true>)
        rollout_cost2<OBJ, MATH, true>(P, A, s_unom, s_trk, splat_state(x0), start, i0, (uint32_t)k0, (uint32_t)b, du_out, Ja, Jb);
    else
        rollout_cost2<OBJ, MATH, false>(P, A, s_unom, s_trk, splat_state(x0), start, i0, (uint32_t)k0, (uint32_t)b, du_out, Ja, Jb, s_xy2, s_z4);
    Ja = sanitize_cost(Ja); Jb = sanitize_cost(Jb);
    *reinterpret_cast<float2*>(A.cost + (size_t)b * P.K + k0) = make_float2(Ja, Jb);

    if (!FUSED) return;

    // ---- block-local softmax partial over the block's 2 blockDim.x samples + last-block combine (mppi_rollout.cuh) ----
    const float Jv[2] = {Ja, Jb};
    block_partial_and_combine_n<MATH, 2>(P, A, b, blockIdx.x, (uint32_t)(2 * blockIdx.x * blockDim.x), Jv, P.T_min, P.T_max,
                                         stored, s_unom, s_red, s_acc, s_pair);
}

// thrust source of the throughput kernel: draw (k, t) in place
template <int MATH>
struct DrawThrust {
    const DevParams& P; const StepArgs& A; const float4* s_unom; uint32_t k, b; float4* du_out;   // du_out: nullptr = not kept
    __device__ __forceinline__ float4 operator()(int t) const
    {
        const float4 un = s_unom[t];
        const float4 T = sample_thrust<MATH>(P, A.rk, k, (uint32_t)t, A.iter, b, un);
        if (du_out)                                        // one coalesced 16-B store per thread
            du_out[(size_t)t * P.K] = make_float4(T.x - un.x, T.y - un.y, T.z - un.z, T.w - un.w);
        return T;
    }
};

// ---------------------------------------------------------------------------------------------
// throughput variant: rollout + cost (+ fused softmax partials and last-block combine)
// grid = (K / blockDim.x, B), one sample per thread
// ---------------------------------------------------------------------------------------------
template <int OBJ, int MATH, bool STORE_DU, bool FUSED>
__global__ void rollout_kernel(const DevParams P, const StepArgs A)
{
    extern __shared__ float4 smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
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

    const State x0 = load_state(A.x0 + 13 * b);
    const int i0 = OBJ == OBJ_CONTOUR ? contour_start_index(P, s_trk, start, x0, s_red) : 0;
    const bool stored = FUSED ? keeps_du<STORE_DU>(A, b) : STORE_DU;
    DrawThrust<MATH> src{P, A, s_unom, (uint32_t)k, (uint32_t)b, stored ? A.du + (size_t)b * N * P.K + k : nullptr};
    const float J = sanitize_cost(rollout_cost<OBJ, MATH>(P, s_trk, x0, start, i0, src));
    A.cost[(size_t)b * P.K + k] = J;

    if (!FUSED) return;

    // block-local softmax partial + last-block combine (mppi_rollout.cuh)
    block_partial_and_combine<MATH>(P, A, b, blockIdx.x, J, P.T_min, P.T_max, s_unom, s_red, s_acc, s_pair, nullptr, nullptr, stored);
}

// ---------------------------------------------------------------------------------------------
// latency variant (fused pipeline only): for a lone controller K = 4096 is 128 warps on 148 SMs,
// and the iteration time is the dependent-issue latency of one warp.  The noise does not depend
// on the state, so it is taken off that critical path:
//   phase 1  all 8 warps of the block draw the clamped thrusts of its 32 C samples for the whole
//            horizon into shared memory (N x (32C+1) float4, rows padded against bank conflicts)
//   phase 2  C consumer warps (one per SM sub-partition) roll the samples out, reading T from smem
//   phase 3  all threads form the block's softmax partial from the thrusts still in shared memory
//            (nothing is re-derived or re-read from HBM), then the last block combines.
// grid = (K / (32 C), B), block = 256 threads.
// ---------------------------------------------------------------------------------------------
struct SmemThrust {
    const float4* col; int row_stride;
    __device__ __forceinline__ float4 operator()(int t) const { return col[t * row_stride]; }
};

constexpr int kLatThreads = 256;

template <int OBJ, int MATH, bool STORE_DU>
__global__ void __launch_bounds__(kLatThreads, 2) rollout_lat_kernel(const DevParams P, const StepArgs A, const int Cflags)
{
    const int C = Cflags & 0xff;                  // rollout warps per block
    const bool split = (Cflags & 0x100) != 0;     // search-contouring: search and cost in warps of their own (host: it fits)
    extern __shared__ float4 smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int b = blockIdx.y, N = P.N;
    const int S = 32 * C, RS = S + 1, lgS = 5 + (C >> 1);             // C in {1, 2, 4}
    const int kbase = blockIdx.x * S;

    float4* s_unom = smem;
    float4* s_trk = smem + N;
    float* s_red = reinterpret_cast<float*>(s_trk + track_f4(P, OBJ));   // 64 floats
    float4* s_T = reinterpret_cast<float4*>(s_red + 64);                 // [N][RS]
    float* s_e = reinterpret_cast<float*>(s_T + (size_t)N * RS);         // 128 floats
    float* s_pair = s_e + 128;

    const int start = A.start[b];
    stage_inputs<OBJ>(P, A, b, start, s_unom, s_trk);
    __syncthreads();

    // ---- phase 1: the whole block draws the noise (eq.(3)) ----
#pragma unroll 2
    for (int idx = tid; idx < N * S; idx += kLatThreads) {
        const int t = idx >> lgS, l = idx & (S - 1);
        const float4 un = s_unom[t];
        const float4 T = sample_thrust<MATH>(P, A.rk, (uint32_t)(kbase + l), (uint32_t)t, A.iter, (uint32_t)b, un);
        s_T[t * RS + l] = T;
        if (STORE_DU)
            A.du[((size_t)b * N + t) * P.K + kbase + l] = make_float4(T.x - un.x, T.y - un.y, T.z - un.z, T.w - un.w);
    }
    const State x0 = load_state(A.x0 + 13 * b);
    const int i0 = OBJ == OBJ_CONTOUR ? contour_start_index(P, s_trk, start, x0, s_red) : 0;
    __syncthreads();

    // ---- phase 2: C warps roll out, one per scheduler ----
    float J = __int_as_float(0x7f800000);
    if (OBJ == OBJ_CONTOUR && split) {
        // Search-based contouring: the windowed nearest-vertex search (33 shared-memory reads and ~300 instructions
        // per step) is as long as the RK4 step itself, and nothing of it feeds back into the dynamics.  So the C
        // rollout warps only integrate and publish (p, |omega|^2) per step; C further warps -- idle otherwise --
        // follow chunk by chunk (mbarriers), search and accumulate the cost.  The two chains overlap instead of adding up.
        float4* s_pos = reinterpret_cast<float4*>(s_pair) + (3 * P.blocks_per_ctrl + 3) / 4;      // [N][S]
        float* s_Jc = reinterpret_cast<float*>(s_pos + (size_t)N * S);                             // [S]
        uint64_t* bar_p = reinterpret_cast<uint64_t*>(s_Jc + S);                                   // [C][chunks]
        const int nch = lat_chunks(N);
        for (int i = tid; i < C * nch; i += kLatThreads) mbar_init(bar_p + i, 32);
        // the candidates once more as register-pair rows for nearest_rot4 (after the barriers, 16-byte aligned)
        float4* s_xy2 = nullptr; float4* s_z4 = nullptr;
        if (contour_pair_f4(P) > 0) {
            const int L = P.P + 2 * P.window + 14;
            const float4* ext = s_trk + 2 * P.P;
            s_xy2 = reinterpret_cast<float4*>(bar_p + 2 * ((C * nch + 1) / 2));
            s_z4 = s_xy2 + L;
            for (int j = tid; j < L; j += kLatThreads) {
                const float4 e0 = ext[j], e1 = ext[min(j + 1, L - 1)], e2 = ext[min(j + 2, L - 1)], e3 = ext[min(j + 3, L - 1)];
                const float far = 1e30f;
                s_xy2[j] = make_float4(e0.x, j + 1 < L ? e1.x : far, e0.y, j + 1 < L ? e1.y : far);
                s_z4[j] = make_float4(e0.z, j + 1 < L ? e1.z : far, j + 2 < L ? e2.z : far, j + 3 < L ? e3.z : far);
            }
        }
        __syncthreads();
        if (warp < C) {
            State x = x0;
            for (int t = 0; t < N; ++t) {
                rk4_step(P, x, s_T[t * RS + tid]);
                s_pos[t * S + tid] = make_float4(x.px, x.py, x.pz, x.ox * x.ox + x.oy * x.oy + x.oz * x.oz);
                if ((t + 1) % kLatChunk == 0 || t == N - 1) mbar_arrive(bar_p + warp * nch + t / kLatChunk);
            }
        } else if (warp < 2 * C) {
            const int w = warp - C, sid = w * 32 + lane;
            ContourCost cc;
            cc.init(P, s_trk, i0, x0);
            float Jc = 0.0f;
            for (int c = 0; c < nch; ++c) {
                mbar_wait(bar_p + w * nch + c, 0);
                const int t1 = min(N, (c + 1) * kLatChunk);
                for (int t = c * kLatChunk; t < t1; ++t) {
                    const float4 q = s_pos[t * S + sid];
                    if (s_xy2) {
                        cc.idx = nearest_rot4(P, s_xy2, s_z4, cc.idx, q.x, q.y, q.z);
                        Jc += cc.step_found(P, s_trk, q.x, q.y, q.z, q.w);
                    } else {
                        Jc += cc.step_at(P, s_trk, q.x, q.y, q.z, q.w);
                    }
                }
            }
            s_Jc[sid] = Jc;
        }
        __syncthreads();
        if (warp < C) {
            J = sanitize_cost(s_Jc[tid]);
            A.cost[(size_t)b * P.K + kbase + tid] = J;
        }
    } else if (warp < C) {
        SmemThrust src{s_T + tid, RS};
        J = sanitize_cost(rollout_cost<OBJ, MATH>(P, s_trk, x0, start, i0, src));
        A.cost[(size_t)b * P.K + kbase + tid] = J;
    }
    const float m = block_min(J, s_red);
    const float e = warp < C ? exp_weight<MATH>((m - J) * P.inv_lambda) : 0.0f;
    const float Zb = block_sum(e, s_red);
    if (warp < C) s_e[tid] = e;
    __syncthreads();

    // ---- phase 3: S[t][i] = sum_l e_l (T_l[t][i] - u_nom[t][i]) from shared memory ----
    float* part = A.partials + ((size_t)b * P.blocks_per_ctrl + blockIdx.x) * P.part_stride;
    for (int j = tid; j < 4 * N; j += kLatThreads) {
        const int t = j >> 2, i = j & 3;
        const float un = reinterpret_cast<const float*>(s_unom)[j];
        const float* row = reinterpret_cast<const float*>(s_T + t * RS) + i;
        float acc = 0.0f;
        for (int l = 0; l < S; ++l) {
            const float el = s_e[l];                      // block-uniform
            if (el != 0.0f) acc = fmaf(el, row[4 * l] - un, acc);
        }
        part[j] = acc;
    }
    if (tid == 0) write_partial_header(P, A, b, blockIdx.x, m, Zb);
    publish_and_combine<MATH, 4>(P, A, b, P.blocks_per_ctrl, s_unom, s_red, s_pair, reinterpret_cast<float*>(s_T));
}

// ---------------------------------------------------------------------------------------------
// TWO_PASS pipeline, second kernel: fused min / exp-weights / normaliser / weighted noise sum
// (eq.(4),(5) PAPER.md:86-95).  grid = (N, B): block (t, b) produces u_new[b][t][0..3]; every
// block re-derives beta and Z from the K costs of its controller (16 KB at K=4096, L2-resident)
// and streams its own K float4 of dU; block t == 0 also writes the weights.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kReduceThreads) reduce_kernel(const DevParams P, const StepArgs A)
{
    __shared__ float s_red[32];
    __shared__ float4 s_red4[kReduceThreads / 32];
    const int t = blockIdx.x, b = blockIdx.y, tid = threadIdx.x;
    const int K = P.K;
    const float* cost = A.cost + (size_t)b * K;

    float m = __int_as_float(0x7f800000);
    for (int k = tid; k < K; k += kReduceThreads) m = fminf(m, cost[k]);
    const float beta = block_min(m, s_red);

    const float4* du = A.du + ((size_t)b * P.N + t) * K;
    float z = 0.0f;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int k = tid; k < K; k += kReduceThreads) {
        const float e = expf((beta - cost[k]) * P.inv_lambda);
        const float4 d = __ldcs(du + k);               // streamed once: evict-first
        z += e;
        acc.x = fmaf(e, d.x, acc.x); acc.y = fmaf(e, d.y, acc.y);
        acc.z = fmaf(e, d.z, acc.z); acc.w = fmaf(e, d.w, acc.w);
    }
    const float Z = block_sum(z, s_red);
    const float invZ = 1.0f / Z;
    acc.x = warp_sum(acc.x); acc.y = warp_sum(acc.y); acc.z = warp_sum(acc.z); acc.w = warp_sum(acc.w);
    if ((tid & 31) == 0) s_red4[tid >> 5] = acc;
    __syncthreads();
    if (tid == 0) {
        float4 s = s_red4[0];
        for (int w = 1; w < kReduceThreads / 32; ++w) {
            s.x += s_red4[w].x; s.y += s_red4[w].y; s.z += s_red4[w].z; s.w += s_red4[w].w;
        }
        const float4 un = reinterpret_cast<const float4*>(A.u_nom)[(size_t)b * P.N + t];
        reinterpret_cast<float4*>(A.u_new)[(size_t)b * P.N + t] =
            make_float4(fmaf(s.x, invZ, un.x), fmaf(s.y, invZ, un.y), fmaf(s.z, invZ, un.z),
                        fmaf(s.w, invZ, un.w));
    }
    if (t == 0)
        for (int k = tid; k < K; k += kReduceThreads)
            A.weights[(size_t)b * K + k] = expf((beta - cost[k]) * P.inv_lambda) * invZ;
}

// ---------------------------------------------------------------------------------------------
// Closed-loop glue: plant RK4 step with u_new[b][0], start-index
// advance, one-step shift of the nominal with its last element repeated [R-14].  One thread
// per controller for the plant, the block's threads share the shift.
// ---------------------------------------------------------------------------------------------
template <int OBJ>
__global__ void sim_kernel(const DevParams P, float* __restrict__ xs, int* __restrict__ start,
                           const float* u_new, float* u_nom_next)
{
    const int b = blockIdx.x;
    const int N = P.N;
    if (threadIdx.x == 0) {
        const int xdim = P.input_model == 1 ? 17 : 13;
        float* xb = xs + xdim * b;
        State x = load_state(xb);
        const float4 T = reinterpret_cast<const float4*>(u_new)[(size_t)b * N];   // thrusts, or thrust rates
        float4 Ts = make_float4(0.f, 0.f, 0.f, 0.f);                               // thrust states (rate model)
        if (P.input_model == 1) Ts = make_float4(xb[13], xb[14], xb[15], xb[16]);
        auto plant = [&]() {
            if (P.input_model == 1) {
                const float4 u = make_float4(fminf(fmaxf(T.x, -P.rate_max), P.rate_max), fminf(fmaxf(T.y, -P.rate_max), P.rate_max),
                                             fminf(fmaxf(T.z, -P.rate_max), P.rate_max), fminf(fmaxf(T.w, -P.rate_max), P.rate_max));
                ThrustDiff D = thrust_diff(Ts);
                rk4_rate_step(P, x, Ts, D, u);
            } else {
                rk4_step(P, x, T);
            }
        };
        if (OBJ == OBJ_GATE) {
            GateCost gc;
            gc.init<0>(P, P.gates, start[b], x);
            plant();
            gc.step<0>(P, P.gates, x);
            start[b] = gc.gate;
        } else if (OBJ == OBJ_TRACK) {
            plant();
            start[b] = min(start[b] + 1, P.M - 1 - N);
        } else {
            plant();
            const int s0 = start[b];
            int i0;
            if (s0 < 0) {
                float best = __int_as_float(0x7f800000);
                i0 = 0;
                for (int i = 0; i < P.P; ++i) {
                    const float4 q = P.path[i];
                    const float dx = x.px - q.x, dy = x.py - q.y, dz = x.pz - q.z;
                    const float d2 = dx * dx + dy * dy + dz * dz;
                    if (d2 < best) { best = d2; i0 = i; }
                }
            } else {
                i0 = ContourCost::nearest(P, P.path, s0, x.px, x.py, x.pz);
            }
            start[b] = i0;
        }
        float* o = xb;
        if (P.input_model == 1) { o[13] = Ts.x; o[14] = Ts.y; o[15] = Ts.z; o[16] = Ts.w; }
        o[0] = x.px; o[1] = x.py; o[2] = x.pz; o[3] = x.qw; o[4] = x.qx; o[5] = x.qy; o[6] = x.qz;
        o[7] = x.vx; o[8] = x.vy; o[9] = x.vz; o[10] = x.ox; o[11] = x.oy; o[12] = x.oz;
    }
    // shift: each thread keeps its source element in a register so that u_nom_next may alias u_new
    const float4* src = reinterpret_cast<const float4*>(u_new) + (size_t)b * N;
    float4* dst = reinterpret_cast<float4*>(u_nom_next) + (size_t)b * N;
    for (int t0 = 0; t0 < N; t0 += blockDim.x) {
        const int t = t0 + threadIdx.x;
        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
        if (t < N) v = src[min(t + 1, N - 1)];
        __syncthreads();
        if (t < N) dst[t] = v;
        __syncthreads();
    }
}

// Plant step under OBJ_CONTOUR_PAPER [R-39]: rows of 19.  The drone takes one rate-model RK4 step with
// u_new[b][0]; the progress states advance by [R-34] with v_new[b][0]; both nominals shift by one step.
// One block per controller; the shifts keep their source in a register so that the outputs may alias
// the inputs.
__global__ void sim_progress_kernel(const DevParams P, float* __restrict__ xs, const float* u_new, float* u_nom_next,
                                    const float* v_new, float* v_nom_next)
{
    const int b = blockIdx.x;
    const int N = P.N;
    if (threadIdx.x == 0) {
        float* xb = xs + 19 * b;
        State x = load_state(xb);
        float4 Ts = make_float4(xb[13], xb[14], xb[15], xb[16]);
        const float theta = xb[17], v_theta = xb[18];
        const float4 T = reinterpret_cast<const float4*>(u_new)[(size_t)b * N];
        const float4 u = make_float4(fminf(fmaxf(T.x, -P.rate_max), P.rate_max), fminf(fmaxf(T.y, -P.rate_max), P.rate_max),
                                     fminf(fmaxf(T.z, -P.rate_max), P.rate_max), fminf(fmaxf(T.w, -P.rate_max), P.rate_max));
        const float dv = fminf(fmaxf(v_new[(size_t)b * N], -P.dv_max), P.dv_max);
        ThrustDiff D = thrust_diff(Ts);
        rk4_rate_step(P, x, Ts, D, u);
        float* o = xb;
        o[0] = x.px; o[1] = x.py; o[2] = x.pz; o[3] = x.qw; o[4] = x.qx; o[5] = x.qy; o[6] = x.qz;
        o[7] = x.vx; o[8] = x.vy; o[9] = x.vz; o[10] = x.ox; o[11] = x.oy; o[12] = x.oz;
        o[13] = Ts.x; o[14] = Ts.y; o[15] = Ts.z; o[16] = Ts.w;
        o[17] = fmaf(P.hh2, dv, fmaf(P.dt, v_theta, theta));
        o[18] = fminf(fmaxf(fmaf(P.dt, dv, v_theta), 0.0f), P.v_theta_max);
    }
    const float4* src = reinterpret_cast<const float4*>(u_new) + (size_t)b * N;
    float4* dst = reinterpret_cast<float4*>(u_nom_next) + (size_t)b * N;
    const float* vsrc = v_new + (size_t)b * N;
    float* vdst = v_nom_next + (size_t)b * N;
    __syncthreads();                       // thread 0 has read u_new[0], v_new[0]
    for (int t0 = 0; t0 < N; t0 += blockDim.x) {
        const int t = t0 + threadIdx.x;
        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
        float w = 0.0f;
        if (t < N) { v = src[min(t + 1, N - 1)]; w = vsrc[min(t + 1, N - 1)]; }
        __syncthreads();
        if (t < N) { dst[t] = v; vdst[t] = w; }
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------------
// "In front of the gate" flags of the noise-free rollout of a nominal sequence [R-26]: what the
// temporal gate-switching check of the paper's J_gate (Fig. 2) compares the next
// control iteration against.  front[b][k] = 1 iff n.(p_k - c) < 0 for the start gate, k = 0..N.
// One thread per controller.
// ---------------------------------------------------------------------------------------------
__global__ void front_flags_kernel(const DevParams P, const float* __restrict__ x0, const int* __restrict__ start,
                                   const float* __restrict__ u, int* __restrict__ front)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= P.B) return;
    const float* xb = x0 + (P.input_model == 1 ? 17 : 13) * b;
    State x = load_state(xb);
    float4 Ts = make_float4(0.f, 0.f, 0.f, 0.f);
    if (P.input_model == 1) Ts = make_float4(xb[13], xb[14], xb[15], xb[16]);
    ThrustDiff D = thrust_diff(Ts);
    const int g = wrap_index(start[b], P.G);
    const float4 c = P.gates[4 * g], n = P.gates[4 * g + 1];
    const float4* ub = reinterpret_cast<const float4*>(u) + (size_t)b * P.N;
    int* fb = front + (size_t)b * (P.N + 1);
    for (int k = 0; k <= P.N; ++k) {
        const float s = fmaf(n.z, x.pz - c.z, fmaf(n.y, x.py - c.y, n.x * (x.px - c.x)));
        fb[k] = s < 0.0f ? 1 : 0;
        if (k == P.N) break;
        float4 T = ub[k];
        const float lo = P.input_model == 1 ? -P.rate_max : P.T_min, hi = P.input_model == 1 ? P.rate_max : P.T_max;
        T.x = fminf(fmaxf(T.x, lo), hi); T.y = fminf(fmaxf(T.y, lo), hi);
        T.z = fminf(fmaxf(T.z, lo), hi); T.w = fminf(fmaxf(T.w, lo), hi);
        if (P.input_model == 1) rk4_rate_step(P, x, Ts, D, T);
        else rk4_step(P, x, T);
    }
}

// ---------------------------------------------------------------------------------------------
// host-side dispatch
// ---------------------------------------------------------------------------------------------
typedef void (*RolloutFn)(const DevParams, const StepArgs);

template <int OBJ, int MATH>
static RolloutFn pick2(const LaunchCfg& c)
{
    if (c.packed) {
        if (c.fused) return c.store_du ? rollout2_kernel<OBJ, MATH, true, true> : rollout2_kernel<OBJ, MATH, false, true>;
        return rollout2_kernel<OBJ, MATH, true, false>;
    }
    if (c.fused) return c.store_du ? rollout_kernel<OBJ, MATH, true, true> : rollout_kernel<OBJ, MATH, false, true>;
    return rollout_kernel<OBJ, MATH, true, false>;
}
template <int OBJ>
static RolloutFn pick1(const LaunchCfg& c)
{
    return c.fast_math ? pick2<OBJ, 1>(c) : pick2<OBJ, 0>(c);
}
static RolloutFn pick(const LaunchCfg& c)
{
    switch (c.objective) {
        case OBJ_GATE: return pick1<OBJ_GATE>(c);
        case OBJ_GATE_PAPER: return pick1<OBJ_GATE_PAPER>(c);
        case OBJ_TRACK: return pick1<OBJ_TRACK>(c);
        default: return pick1<OBJ_CONTOUR>(c);
    }
}

typedef void (*LatFn)(const DevParams, const StepArgs, const int);

template <int OBJ>
static LatFn pick_lat1(const LaunchCfg& c)
{
    if (c.fast_math) return c.store_du ? rollout_lat_kernel<OBJ, 1, true> : rollout_lat_kernel<OBJ, 1, false>;
    return c.store_du ? rollout_lat_kernel<OBJ, 0, true> : rollout_lat_kernel<OBJ, 0, false>;
}
static LatFn pick_lat(const LaunchCfg& c)
{
    switch (c.objective) {
        case OBJ_GATE: return pick_lat1<OBJ_GATE>(c);
        case OBJ_GATE_PAPER: return pick_lat1<OBJ_GATE_PAPER>(c);
        case OBJ_TRACK: return pick_lat1<OBJ_TRACK>(c);
        default: return pick_lat1<OBJ_CONTOUR>(c);
    }
}

typedef void (*PipeFn)(const DevParams, const StepArgs);
template <int OBJ>
static PipeFn pick_pipe1(const LaunchCfg& c)
{
    if (c.fast_math) return c.store_du ? rollout_pipe_kernel<OBJ, 1, true> : rollout_pipe_kernel<OBJ, 1, false>;
    return c.store_du ? rollout_pipe_kernel<OBJ, 0, true> : rollout_pipe_kernel<OBJ, 0, false>;
}
static PipeFn pick_pipe(const LaunchCfg& c)
{
    switch (c.objective) {
        case OBJ_GATE: return pick_pipe1<OBJ_GATE>(c);
        case OBJ_GATE_PAPER: return pick_pipe1<OBJ_GATE_PAPER>(c);
        case OBJ_TRACK: return pick_pipe1<OBJ_TRACK>(c);
        default: return pick_pipe1<OBJ_CONTOUR>(c);
    }
}

const void* rollout_kernel_ptr(const LaunchCfg& c)
{
    if (c.rate) return rate_kernel_ptr(c);
    if (c.scan) return scan_kernel_ptr(c);
    if (c.pipe) return reinterpret_cast<const void*>(pick_pipe(c));
    return c.lat_consumers > 0 ? reinterpret_cast<const void*>(pick_lat(c)) : reinterpret_cast<const void*>(pick(c));
}
const void* reduce_kernel_ptr() { return reinterpret_cast<const void*>(reduce_kernel); }
const void* sim_kernel_ptr() { return reinterpret_cast<const void*>(sim_kernel<OBJ_GATE>); }

cudaError_t launch_rollout(const DevParams& P, const StepArgs& A, const LaunchCfg& c, cudaStream_t s, bool pdl)
{
    const dim3 grid(P.blocks_per_ctrl, P.B), block(c.block_threads);
    if (c.rate) return launch_rate(P, A, c, s);
    if (c.scan) return launch_scan(P, A, c, s, pdl);
    if (c.pipe && pdl) {
        // programmatic dependent launch: this kernel may start before the previous kernel of the stream has finished;
        // it orders itself with griddepcontrol.wait (StepArgs::pdl bit 0 must be set)
        cudaLaunchConfig_t lc;
        memset(&lc, 0, sizeof lc);
        lc.gridDim = grid; lc.blockDim = block; lc.dynamicSmemBytes = c.smem_bytes; lc.stream = s;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        lc.attrs = at; lc.numAttrs = 1;
        return cudaLaunchKernelEx(&lc, pick_pipe(c), P, A);
    }
    if (c.pipe) pick_pipe(c)<<<grid, block, c.smem_bytes, s>>>(P, A);
    else if (c.lat_consumers > 0) pick_lat(c)<<<grid, block, c.smem_bytes, s>>>(P, A, c.lat_consumers | (c.lat_split << 8));
    else pick(c)<<<grid, block, c.smem_bytes, s>>>(P, A);
    return cudaGetLastError();
}

cudaError_t launch_reduce(const DevParams& P, const StepArgs& A, cudaStream_t s)
{
    reduce_kernel<<<dim3(P.N, P.B), kReduceThreads, 0, s>>>(P, A);
    return cudaGetLastError();
}

cudaError_t launch_sim(const DevParams& P, int objective, float* x, int* start, const float* u_new,
                       float* u_nom_next, cudaStream_t s)
{
    const int threads = 64;
    if (objective == OBJ_GATE || objective == OBJ_GATE_PAPER)       // the plant's gate advance is geometric
        sim_kernel<OBJ_GATE><<<P.B, threads, 0, s>>>(P, x, start, u_new, u_nom_next);
    else if (objective == OBJ_TRACK) sim_kernel<OBJ_TRACK><<<P.B, threads, 0, s>>>(P, x, start, u_new, u_nom_next);
    else sim_kernel<OBJ_CONTOUR><<<P.B, threads, 0, s>>>(P, x, start, u_new, u_nom_next);
    return cudaGetLastError();
}

cudaError_t launch_sim_progress(const DevParams& P, float* x, const float* u_new, float* u_nom_next,
                                const float* v_new, float* v_nom_next, cudaStream_t s)
{
    sim_progress_kernel<<<P.B, 64, 0, s>>>(P, x, u_new, u_nom_next, v_new, v_nom_next);
    return cudaGetLastError();
}

cudaError_t launch_front(const DevParams& P, const float* x0, const int* start, const float* u, int* front,
                         cudaStream_t s)
{
    front_flags_kernel<<<(P.B + 63) / 64, 64, 0, s>>>(P, x0, start, u, front);
    return cudaGetLastError();
}

}  // namespace mppi
