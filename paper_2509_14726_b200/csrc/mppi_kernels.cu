// mppi_kernels.cu -- the sm_100a kernels of the MPPI hot path.
//
//   rollout_kernel<OBJ, MATH, STORE_DU, FUSED>   SURVEY.md 8(a) steps 1-4 (+5-7 when FUSED)
//   reduce_kernel                                steps 5-7 of the TWO_PASS pipeline
//   sim_kernel                                   step 8 (closed-loop glue)
//
// Thread mapping: one sample per thread, block = blockDim.x consecutive samples of ONE
// controller, grid = (K / blockDim.x, B).  No tensor cores: nothing here is a contraction.
#include "mppi_cost.cuh"
#include "mppi_internal.h"

namespace mppi {

constexpr unsigned kFull = 0xffffffffu;

__device__ __forceinline__ float warp_min(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fminf(v, __shfl_xor_sync(kFull, v, o));
    return v;
}
__device__ __forceinline__ float warp_sum(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    return v;
}

template <int MATH>
__device__ __forceinline__ float exp_weight(float x)   // exp(x), x <= 0
{
    return MATH == 0 ? expf(x) : __expf(x);
}

// block-wide min / sum over blockDim.x threads through s_red[0..31]; every thread gets the result
__device__ __forceinline__ float block_min(float v, float* s_red)
{
    v = warp_min(v);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = v;
    __syncthreads();
    const int nw = blockDim.x >> 5;
    float r = s_red[0];
    for (int w = 1; w < nw; ++w) r = fminf(r, s_red[w]);
    return r;
}
__device__ __forceinline__ float block_sum(float v, float* s_red)
{
    v = warp_sum(v);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = v;
    __syncthreads();
    const int nw = blockDim.x >> 5;
    float r = s_red[0];
    for (int w = 1; w < nw; ++w) r += s_red[w];      // fixed order: deterministic
    return r;
}

// Shared-memory carve-up of the rollout kernel (units: float4).
//   [0, N)                         nominal thrusts u_nom[b]
//   [N, N + trk)                   track data of the objective
//   then 16 float4                 reduction scratch (64 floats)
//   FUSED: nwarps * N float4       per-warp weighted-noise accumulators
//   FUSED: ceil(nblk/4) float4     per-block rescale factors of the last-block combine
__host__ __device__ inline int track_f4(const DevParams& P, int objective)
{
    return objective == OBJ_GATE ? 4 * P.G : objective == OBJ_TRACK ? 4 * (P.N + 1) : 2 * P.P;
}

size_t rollout_smem_bytes(const DevParams& P, const LaunchCfg& c)
{
    size_t f4 = (size_t)P.N + track_f4(P, c.objective) + 16;
    if (c.fused) f4 += (size_t)(c.block_threads / 32) * P.N + (P.blocks_per_ctrl + 3) / 4;
    return f4 * sizeof(float4);
}

// ---------------------------------------------------------------------------------------------
// rollout + cost (+ fused softmax partials and last-block combine)
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
    float* s_scale = reinterpret_cast<float*>(s_acc + (blockDim.x >> 5) * N);

    // ---- stage the nominal sequence and the track in shared memory ----
    const int start = A.start[b];
    {
        const float4* un = reinterpret_cast<const float4*>(A.u_nom) + (size_t)b * N;
        for (int t = tid; t < N; t += blockDim.x) s_unom[t] = un[t];
        if (OBJ == OBJ_GATE) {
            for (int i = tid; i < 4 * P.G; i += blockDim.x) s_trk[i] = P.gates[i];
        } else if (OBJ == OBJ_TRACK) {
            const int t0 = min(max(start, 0), P.M - 1 - N);
            for (int i = tid; i < 4 * (N + 1); i += blockDim.x) s_trk[i] = P.ref[4 * t0 + i];
        } else {
            for (int i = tid; i < 2 * P.P; i += blockDim.x) s_trk[i] = P.path[i];
        }
    }
    __syncthreads();

    State x = load_state(A.x0 + 13 * b);
    float J = 0.0f;
    GateCost gc;
    ContourCost cc;
    if (OBJ == OBJ_GATE) gc.init<MATH>(P, s_trk, start, x);
    if (OBJ == OBJ_CONTOUR) {
        int i0;
        if (start < 0) {
            // global nearest vertex, block-cooperative; ties -> smallest index (scan order)
            float best = __int_as_float(0x7f800000);
            int ib = 0x7fffffff;
            for (int i = tid; i < P.P; i += blockDim.x) {
                const float4 q = s_trk[2 * i];
                const float dx = x.px - q.x, dy = x.py - q.y, dz = x.pz - q.z;
                const float d2 = dx * dx + dy * dy + dz * dz;
                if (d2 < best) { best = d2; ib = i; }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const float ob = __shfl_xor_sync(kFull, best, o);
                const int oi = __shfl_xor_sync(kFull, ib, o);
                if (ob < best || (ob == best && oi < ib)) { best = ob; ib = oi; }
            }
            if (lane == 0) { s_red[warp] = best; reinterpret_cast<int*>(s_red)[32 + warp] = ib; }
            __syncthreads();
            best = s_red[0]; ib = reinterpret_cast<int*>(s_red)[32];
            for (int w = 1; w < (int)(blockDim.x >> 5); ++w) {
                const float ob = s_red[w];
                const int oi = reinterpret_cast<int*>(s_red)[32 + w];
                if (ob < best || (ob == best && oi < ib)) { best = ob; ib = oi; }
            }
            i0 = ib;
            __syncthreads();
        } else {
            const int centre = P.closed ? wrap_index(start, P.P) : min(max(start, 0), P.P - 1);
            i0 = ContourCost::nearest(P, s_trk, centre, x.px, x.py, x.pz);
        }
        cc.init(s_trk, i0, x);
    }

    // ---- the horizon: noise -> clamp -> RK4 -> cost, all in registers (Alg. 1 lines 6-13) ----
    float4* du_out = STORE_DU ? A.du + (size_t)b * N * P.K + k : nullptr;
    for (int t = 0; t < N; ++t) {
        const float4 un = s_unom[t];
        const float4 T = sample_thrust<MATH>(P, A.rk, (uint32_t)k, (uint32_t)t, A.iter, (uint32_t)b, un);
        if (STORE_DU)                                      // one coalesced 16-B store per thread
            du_out[(size_t)t * P.K] = make_float4(T.x - un.x, T.y - un.y, T.z - un.z, T.w - un.w);
        if (OBJ == OBJ_TRACK) J += track_stage(P, s_trk + 4 * t, x, T);
        rk4_step(P, x, T);
        if (OBJ == OBJ_GATE) gc.step<MATH>(P, s_trk, x);
        if (OBJ == OBJ_CONTOUR) J += cc.step(P, s_trk, x);
    }
    if (OBJ == OBJ_GATE) J = gc.finish<MATH>(P, s_trk, x);
    if (OBJ == OBJ_TRACK) J += track_state_term(P, s_trk + 4 * N, x);
    A.cost[(size_t)b * P.K + k] = J;

    if (!FUSED) return;

    // ---- block-local softmax partial (online-softmax form of eq.(4),(5)) ----
    // m = min_k J, e_k = exp(-(J_k - m)/lambda), Z = sum e_k, S[t] = sum_k e_k dU_k[t].
    // dU is not stored anywhere: for the samples with e_k > 0 it is re-derived from the
    // counter-based stream, the warp's lanes spread over the horizon steps.
    const float m = block_min(J, s_red);
    const float e = exp_weight<MATH>((m - J) * P.inv_lambda);
    const float Zb = block_sum(e, s_red);
    {
        const unsigned contrib = __ballot_sync(kFull, e > 0.0f);
        const uint32_t kbase = (uint32_t)(blockIdx.x * blockDim.x + warp * 32);
        for (int t0 = 0; t0 < N; t0 += 32) {
            const int t = t0 + lane;
            const float4 un = t < N ? s_unom[t] : make_float4(0.f, 0.f, 0.f, 0.f);
            float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
            unsigned mm = contrib;
            while (mm) {
                const int l = __ffs(mm) - 1;
                mm &= mm - 1;
                const float el = __shfl_sync(kFull, e, l);
                const float4 T = sample_thrust<MATH>(P, A.rk, kbase + l, (uint32_t)t, A.iter, (uint32_t)b, un);
                acc.x = fmaf(el, T.x - un.x, acc.x); acc.y = fmaf(el, T.y - un.y, acc.y);
                acc.z = fmaf(el, T.z - un.z, acc.z); acc.w = fmaf(el, T.w - un.w, acc.w);
            }
            if (t < N) s_acc[warp * N + t] = acc;
        }
    }
    __syncthreads();
    const int nw = blockDim.x >> 5;
    const int stride = 4 * N + 4;
    float* part = A.partials + ((size_t)b * P.blocks_per_ctrl + blockIdx.x) * stride;
    for (int j = tid; j < 4 * N; j += blockDim.x) {
        float s = 0.0f;
        for (int w = 0; w < nw; ++w) s += reinterpret_cast<const float*>(s_acc)[w * 4 * N + j];
        part[j] = s;
    }
    if (tid == 0) { part[4 * N] = m; part[4 * N + 1] = Zb; }

    // ---- last block of this controller combines the partials ("threadfence reduction") ----
    __threadfence();
    __syncthreads();
    if (tid == 0) {
        const unsigned ticket = atomicAdd(&A.counters[b], 1u);
        reinterpret_cast<int*>(s_red)[40] = (ticket == (unsigned)(P.blocks_per_ctrl - 1));
    }
    __syncthreads();
    if (!reinterpret_cast<int*>(s_red)[40]) return;
    __threadfence();

    const int nb = P.blocks_per_ctrl;
    const float* pb = A.partials + (size_t)b * nb * stride;
    float bm = __int_as_float(0x7f800000);
    for (int j = tid; j < nb; j += blockDim.x) bm = fminf(bm, __ldcg(pb + (size_t)j * stride + 4 * N));
    const float beta = block_min(bm, s_red);
    float zz = 0.0f;
    for (int j = tid; j < nb; j += blockDim.x) {
        const float sc = exp_weight<MATH>((beta - __ldcg(pb + (size_t)j * stride + 4 * N)) * P.inv_lambda);
        s_scale[j] = sc;
        zz = fmaf(__ldcg(pb + (size_t)j * stride + 4 * N + 1), sc, zz);
    }
    const float Z = block_sum(zz, s_red);      // also orders the s_scale writes before the reads
    const float invZ = 1.0f / Z;
    for (int j = tid; j < 4 * N; j += blockDim.x) {
        float acc = 0.0f;
        for (int q = 0; q < nb; ++q) acc = fmaf(__ldcg(pb + (size_t)q * stride + j), s_scale[q], acc);
        A.u_new[(size_t)b * 4 * N + j] = fmaf(acc, invZ, reinterpret_cast<const float*>(s_unom)[j]);
    }
    for (int kk = tid; kk < P.K; kk += blockDim.x) {
        const float Jk = __ldcg(A.cost + (size_t)b * P.K + kk);
        A.weights[(size_t)b * P.K + kk] = exp_weight<MATH>((beta - Jk) * P.inv_lambda) * invZ;
    }
    if (tid == 0) A.counters[b] = 0u;          // ready for the next launch
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
        State x = load_state(xs + 13 * b);
        const float4 T = reinterpret_cast<const float4*>(u_new)[(size_t)b * N];
        if (OBJ == OBJ_GATE) {
            GateCost gc;
            gc.init<0>(P, P.gates, start[b], x);
            rk4_step(P, x, T);
            gc.step<0>(P, P.gates, x);
            start[b] = gc.gate;
        } else if (OBJ == OBJ_TRACK) {
            rk4_step(P, x, T);
            start[b] = min(start[b] + 1, P.M - 1 - N);
        } else {
            rk4_step(P, x, T);
            const int s0 = start[b];
            int i0;
            if (s0 < 0) {
                float best = __int_as_float(0x7f800000);
                i0 = 0;
                for (int i = 0; i < P.P; ++i) {
                    const float4 q = P.path[2 * i];
                    const float dx = x.px - q.x, dy = x.py - q.y, dz = x.pz - q.z;
                    const float d2 = dx * dx + dy * dy + dz * dz;
                    if (d2 < best) { best = d2; i0 = i; }
                }
            } else {
                i0 = ContourCost::nearest(P, P.path, s0, x.px, x.py, x.pz);
            }
            start[b] = i0;
        }
        float* o = xs + 13 * b;
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

// ---------------------------------------------------------------------------------------------
// host-side dispatch
// ---------------------------------------------------------------------------------------------
typedef void (*RolloutFn)(const DevParams, const StepArgs);

template <int OBJ, int MATH>
static RolloutFn pick2(const LaunchCfg& c)
{
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
        case OBJ_TRACK: return pick1<OBJ_TRACK>(c);
        default: return pick1<OBJ_CONTOUR>(c);
    }
}

const void* rollout_kernel_ptr(const LaunchCfg& c) { return reinterpret_cast<const void*>(pick(c)); }
const void* reduce_kernel_ptr() { return reinterpret_cast<const void*>(reduce_kernel); }
const void* sim_kernel_ptr() { return reinterpret_cast<const void*>(sim_kernel<OBJ_GATE>); }

cudaError_t launch_rollout(const DevParams& P, const StepArgs& A, const LaunchCfg& c, cudaStream_t s)
{
    const dim3 grid(P.blocks_per_ctrl, P.B), block(c.block_threads);
    pick(c)<<<grid, block, c.smem_bytes, s>>>(P, A);
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
    if (objective == OBJ_GATE) sim_kernel<OBJ_GATE><<<P.B, threads, 0, s>>>(P, x, start, u_new, u_nom_next);
    else if (objective == OBJ_TRACK) sim_kernel<OBJ_TRACK><<<P.B, threads, 0, s>>>(P, x, start, u_new, u_nom_next);
    else sim_kernel<OBJ_CONTOUR><<<P.B, threads, 0, s>>>(P, x, start, u_new, u_nom_next);
    return cudaGetLastError();
}

}  // namespace mppi
