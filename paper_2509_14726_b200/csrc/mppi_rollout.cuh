// mppi_rollout.cuh -- device functions shared by the two rollout kernels (throughput and latency
// variants): block reductions, shared-memory staging, the horizon loop, and the last-block
// combine of the fused softmax update.
#pragma once
#include "mppi_cost.cuh"

namespace mppi {

constexpr unsigned kFull = 0xffffffffu;

// minimum over the warp: ONE instruction on sm_100a (redux.sync.min.f32 -> CREDUX.MIN.F32, result in a uniform
// register) instead of five shuffle + FMNMX rounds; the minimum is exact, so nothing else changes.  NaN inputs are
// ignored, as by fminf (costs are sanitised before they get here).
__device__ __forceinline__ float warp_min(float v)
{
    float r;
    asm volatile("redux.sync.min.f32 %0, %1, 0xffffffff;" : "=f"(r) : "f"(v));
    return r;
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
    return MATH == 0 ? expf(x) : mufu_ex2(x * 1.4426950408889634f);
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

__host__ __device__ inline int track_f4(const DevParams& P, int objective)
{
    return objective == OBJ_GATE ? 4 * P.G
         : objective == OBJ_GATE_PAPER ? 4 * P.G + (P.N + 4) / 4      // gates + N+1 previous-iteration flags
         : objective == OBJ_TRACK ? 4 * (P.N + 1)
         : objective == OBJ_CONTOUR ? 3 * P.P + 2 * P.window + 14       // path + padded copy of the points (nearest_ext; 2 kExtPad)
         : 2 * P.P;                                                    // the paper's contouring: the path
}

// Stage the nominal sequence of controller b and the objective's track data in shared memory.
__device__ __forceinline__ void stage_nominal(const DevParams& P, const StepArgs& A, int b, float4* s_unom)
{
    const float4* un = reinterpret_cast<const float4*>(A.u_nom) + (size_t)b * P.N;
    for (int t = threadIdx.x; t < P.N; t += blockDim.x) s_unom[t] = un[t];
}
template <int OBJ>
__device__ __forceinline__ void stage_track(const DevParams& P, const StepArgs& A, int b, int start, float4* s_trk);
template <int OBJ>
__device__ __forceinline__ void stage_inputs(const DevParams& P, const StepArgs& A, int b, int start,
                                             float4* s_unom, float4* s_trk)
{
    stage_nominal(P, A, b, s_unom);
    stage_track<OBJ>(P, A, b, start, s_trk);
}
// The objective's track data only (constant inputs: nothing a previous kernel of the stream writes).
template <int OBJ>
__device__ __forceinline__ void stage_track(const DevParams& P, const StepArgs& A, int b, int start, float4* s_trk)
{
    const int tid = threadIdx.x, N = P.N;
    if (OBJ == OBJ_GATE) {
        for (int i = tid; i < 4 * P.G; i += blockDim.x) s_trk[i] = P.gates[i];
    } else if (OBJ == OBJ_GATE_PAPER) {
        for (int i = tid; i < 4 * P.G; i += blockDim.x) s_trk[i] = P.gates[i];
        int* s_front = reinterpret_cast<int*>(s_trk + 4 * P.G);
        for (int i = tid; i <= N; i += blockDim.x) s_front[i] = A.prev_front ? A.prev_front[(size_t)b * (N + 1) + i] : 1;
    } else if (OBJ == OBJ_TRACK) {
        const int t0 = min(max(start, 0), P.M - 1 - N);
        for (int i = tid; i < 4 * (N + 1); i += blockDim.x) s_trk[i] = P.ref[4 * t0 + i];
    } else {
        for (int i = tid; i < 2 * P.P; i += blockDim.x) s_trk[i] = P.path[i];
        if (OBJ == OBJ_CONTOUR) {      // padded copy of the points for the windowed search (ContourCost::nearest_ext)
            float4* ext = s_trk + 2 * P.P;
            for (int j = tid; j < P.P + 2 * P.window + 14; j += blockDim.x) {
                int i = j - P.window - 7;                        // ContourCost::kExtPad entries in front and behind
                if (P.closed) i = i < 0 ? i + P.P : (i >= P.P ? i - P.P : i);
                ext[j] = (i >= 0 && i < P.P) ? P.path[i] : make_float4(1e30f, 1e30f, 1e30f, 0.0f);
            }
        }
    }
}

// Contouring: initial path index of the block (all samples share x0).  start < 0: global nearest
// vertex, block-cooperative, ties -> smallest index (= the oracle's scan order); otherwise the
// windowed search around the hint.  Every thread of the block must call this.
__device__ __forceinline__ int contour_start_index(const DevParams& P, const float4* s_path, int start,
                                                   const State& x, float* s_red)
{
    if (start >= 0) {
        const int centre = P.closed ? wrap_index(start, P.P) : min(max(start, 0), P.P - 1);
        return ContourCost::nearest_smem(P, s_path, centre, x.px, x.py, x.pz);
    }
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    float best = __int_as_float(0x7f800000);
    int ib = 0x7fffffff;
    for (int i = tid; i < P.P; i += blockDim.x) {
        const float4 q = s_path[i];
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
    int* s_idx = reinterpret_cast<int*>(s_red) + 32;
    if (lane == 0) { s_red[warp] = best; s_idx[warp] = ib; }
    __syncthreads();
    best = s_red[0]; ib = s_idx[0];
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) {
        const float ob = s_red[w];
        const int oi = s_idx[w];
        if (ob < best || (ob == best && oi < ib)) { best = ob; ib = oi; }
    }
    __syncthreads();
    return ib;
}

// The horizon of one sample: thrust -> RK4 -> cost, all in registers (Alg. 1 lines 6-13).
// `thrust(t)` yields the clamped rotor thrusts of step t (drawn in place or read from smem).
template <int OBJ, int MATH, class Thrust>
__device__ __forceinline__ float rollout_cost(const DevParams& P, const float4* s_trk, State x, int start,
                                              int contour_i0, Thrust thrust)
{
    const int N = P.N;
    float J = 0.0f;
    GateCost gc;
    GatePaperCost gp;
    ContourCost cc;
    const int* s_front = reinterpret_cast<const int*>(s_trk + 4 * P.G);      // OBJ_GATE_PAPER only
    if (OBJ == OBJ_GATE) gc.init<MATH>(P, s_trk, start, x);
    if (OBJ == OBJ_GATE_PAPER) gp.init(P, s_trk, start, x);
    if (OBJ == OBJ_CONTOUR) cc.init(P, s_trk, contour_i0, x);
    for (int t = 0; t < N; ++t) {
        const float4 T = thrust(t);
        if (OBJ == OBJ_TRACK) J += track_stage(P, s_trk + 4 * t, x, T);
        rk4_step(P, x, T);
        if (OBJ == OBJ_GATE) gc.step<MATH>(P, s_trk, x);
        if (OBJ == OBJ_GATE_PAPER) gp.step(P, s_trk, s_front, x, t);
        if (OBJ == OBJ_CONTOUR) J += cc.step(P, s_trk, x);
    }
    if (OBJ == OBJ_GATE) J = gc.finish<MATH>(P, s_trk, x);
    if (OBJ == OBJ_GATE_PAPER) J = gp.finish(P);
    if (OBJ == OBJ_TRACK) J += track_state_term(P, s_trk + 4 * N, x);
    return J;
}

// header of a partial: (m, Z) of block `chunk` of controller b, in an array of its own (8 bytes per partial, contiguous
// per controller) so that the combining block reads all headers of a controller in nb / 16 cache lines.
__device__ __forceinline__ void write_partial_header(const DevParams& P, const StepArgs& A, const int b, const int chunk,
                                                     const float m, const float Zb)
{
    A.headers[(size_t)b * P.blocks_per_ctrl + chunk] = make_float2(m, Zb);
}

// Fused softmax update, first half, for kernels with one sample per thread: the block's online-softmax
// partial  m = min_k J, e_k = exp(-(J_k - m)/lambda), Z = sum e_k, S[t] = sum_k e_k dU_k[t]  (eq.(4),(5)).
// dU is not stored anywhere: for the samples with e_k > 0 it is re-derived from the counter-based
// stream (inputs clamped to [lo, hi] as in the rollout), the warp's lanes spread over the horizon
// steps.  Then publish_and_combine.  All threads of the block must call this.
template <int MATH, int ROWS = 2>
__device__ __forceinline__ void publish_and_combine(const DevParams& P, const StepArgs& A, int b, int nb,
                                                    const float4* s_unom, float* s_red, float* s_pair, float* s_work,
                                                    const float* s_vnom = nullptr);
template <int MATH>
__device__ __forceinline__ float sample_progress_accel(const DevParams& P, const uint32_t (&rk)[20], uint32_t k,
                                                       uint32_t t, uint32_t iter, uint32_t b, const float vn);
// The warp's share of S[t] = sum_k e_k dU_k[t] (eq.(5)) for kernels that hold SPT samples per lane:
// lane l owns samples kbase + SPT l + h with weights e[h].  Two ways, both exact:
//   sparse  the perturbations are RE-DERIVED from the counter-based stream for the samples with e > 0 only, the
//           lanes spread over the horizon steps -- nearly free when the softmax is one-hot (every config of
//           BASELINE.json, the paper's lambda = 0.01), but the whole noise stream again when most samples count;
//   dense   when this launch also STORED dU (du_ctrl != nullptr; see StepArgs::hint) and enough samples of the warp
//           count: every lane reads its own rows back (L2 hits for the most part: the block wrote them during the
//           rollout), and eight steps at a time are summed over the lanes by a transposed butterfly (7 + 2 shuffle
//           rounds per component instead of 5 per step).
// s_acc_row: N float4 of this warp.  s_vnom / s_acc5_row (OBJ_CONTOUR_PAPER only, else nullptr): the nominal of the
// fifth sampled input and its accumulator row; that column is always re-derived.
__device__ __forceinline__ float4 shfl_xor4(const float4 v, const int m)
{
    return make_float4(__shfl_xor_sync(kFull, v.x, m), __shfl_xor_sync(kFull, v.y, m), __shfl_xor_sync(kFull, v.z, m),
                       __shfl_xor_sync(kFull, v.w, m));
}
__device__ __forceinline__ float4 add4(const float4 a, const float4 b) { return make_float4(a.x + b.x, a.y + b.y, a.z + b.z, a.w + b.w); }

template <int MATH, int SPT>
__device__ __forceinline__ void warp_noise_partial(const DevParams& P, const StepArgs& A, const int b, const uint32_t kbase,
                                                   const float (&e)[SPT], const float lo, const float hi,
                                                   const float4* s_unom, float4* s_acc_row, const float4* du_ctrl,
                                                   const float* s_vnom = nullptr, float* s_acc5_row = nullptr)
{
    const int lane = threadIdx.x & 31, N = P.N;
    unsigned contrib[SPT];
    int count = 0;
#pragma unroll
    for (int h = 0; h < SPT; ++h) { contrib[h] = __ballot_sync(kFull, e[h] > 0.0f); count += __popc(contrib[h]); }
    // instruction estimate per lane: sparse ~ 85 per (contributing sample, pass of 32 steps); dense ~ 5 SPT + 16 per step
    if (du_ctrl && !s_vnom && count * ((N + 31) >> 5) * 85 > N * (5 * SPT + 16)) {
        const float4* mine = du_ctrl + kbase + SPT * lane;
        const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4;
        const int t_off = (b4 ? 4 : 0) + (b3 ? 2 : 0) + (b2 ? 1 : 0);
        for (int t0 = 0; t0 < N; t0 += 8) {
            float4 v[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                v[j] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (t0 + j < N) {
#pragma unroll
                    for (int h = 0; h < SPT; ++h) {
                        const float4 d = mine[(size_t)(t0 + j) * P.K + h];
                        v[j].x = fmaf(e[h], d.x, v[j].x); v[j].y = fmaf(e[h], d.y, v[j].y);
                        v[j].z = fmaf(e[h], d.z, v[j].z); v[j].w = fmaf(e[h], d.w, v[j].w);
                    }
                }
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const float4 send = b4 ? v[j] : v[j + 4], keep = b4 ? v[j + 4] : v[j];
                v[j] = add4(keep, shfl_xor4(send, 16));
            }
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const float4 send = b3 ? v[j] : v[j + 2], keep = b3 ? v[j + 2] : v[j];
                v[j] = add4(keep, shfl_xor4(send, 8));
            }
            {
                const float4 send = b2 ? v[0] : v[1], keep = b2 ? v[1] : v[0];
                v[0] = add4(keep, shfl_xor4(send, 4));
            }
            v[0] = add4(v[0], shfl_xor4(v[0], 2));
            v[0] = add4(v[0], shfl_xor4(v[0], 1));
            if ((lane & 3) == 0 && t0 + t_off < N) s_acc_row[t0 + t_off] = v[0];
        }
        return;
    }
    for (int t0 = 0; t0 < N; t0 += 32) {
        const int t = t0 + lane;
        const float4 un = t < N ? s_unom[t] : make_float4(0.f, 0.f, 0.f, 0.f);
        const float vn = (s_vnom && t < N) ? s_vnom[t] : 0.0f;
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
        float acc5 = 0.0f;
#pragma unroll
        for (int h = 0; h < SPT; ++h) {
            unsigned mm = contrib[h];
            while (mm) {
                const int l = __ffs(mm) - 1;
                mm &= mm - 1;
                const float el = __shfl_sync(kFull, e[h], l);
                const uint32_t k = kbase + (uint32_t)(SPT * l + h);
                const float4 T = sample_input<MATH>(P, A.rk, k, (uint32_t)t, A.iter, (uint32_t)b, un, lo, hi);
                acc.x = fmaf(el, T.x - un.x, acc.x); acc.y = fmaf(el, T.y - un.y, acc.y);
                acc.z = fmaf(el, T.z - un.z, acc.z); acc.w = fmaf(el, T.w - un.w, acc.w);
                if (s_vnom)
                    acc5 = fmaf(el, sample_progress_accel<MATH>(P, A.rk, k, (uint32_t)t, A.iter, (uint32_t)b, vn) - vn, acc5);
            }
        }
        if (t < N) { s_acc_row[t] = acc; if (s_vnom) s_acc5_row[t] = acc5; }
    }
}

// Does this launch keep dU of controller b?  Always when the kernel was built for it (two-pass pipeline, store_noise);
// in the fused pipeline also when the previous iteration's combine found many samples carrying weight (StepArgs::hint).
template <bool STORE_DU>
__device__ __forceinline__ bool keeps_du(const StepArgs& A, const int b)
{
    return STORE_DU || (A.hint != nullptr && A.du != nullptr && A.hint[b] != 0u);
}

// Block partial for kernels with SPT samples per thread: block minimum, weights, warp sums (warp_noise_partial), sum
// over the warps, the partial's (m, Z) header, then publish_and_combine.  All threads of the block must call this.
// chunk: index of this block within its controller; kblock: its first sample.
template <int MATH, int SPT>
__device__ __forceinline__ void block_partial_and_combine_n(const DevParams& P, const StepArgs& A, const int b,
                                                            const int chunk, const uint32_t kblock, const float (&J)[SPT],
                                                            const float lo, const float hi, const bool stored,
                                                            const float4* s_unom, float* s_red, float4* s_acc, float* s_pair,
                                                            const float* s_vnom = nullptr, float* s_acc5 = nullptr)
{
    const int tid = threadIdx.x, warp = tid >> 5, N = P.N;
    float jm = J[0];
#pragma unroll
    for (int h = 1; h < SPT; ++h) jm = fminf(jm, J[h]);
    const float m = block_min(jm, s_red);
    float e[SPT], es = 0.0f;
#pragma unroll
    for (int h = 0; h < SPT; ++h) { e[h] = exp_weight<MATH>((m - J[h]) * P.inv_lambda); es += e[h]; }
    const float Zb = block_sum(es, s_red);
    warp_noise_partial<MATH, SPT>(P, A, b, kblock + (uint32_t)(warp * 32 * SPT), e, lo, hi, s_unom, s_acc + warp * N,
                                  stored ? A.du + (size_t)b * N * P.K : nullptr, s_vnom, s_acc5 ? s_acc5 + warp * N : nullptr);
    __syncthreads();
    const int nw = blockDim.x >> 5;
    float* part = A.partials + ((size_t)b * P.blocks_per_ctrl + chunk) * P.part_stride;
    for (int j = tid; j < 4 * N; j += blockDim.x) {
        float s = 0.0f;
        for (int w = 0; w < nw; ++w) s += reinterpret_cast<const float*>(s_acc)[w * 4 * N + j];
        part[j] = s;
    }
    if (s_vnom)
        for (int t = tid; t < N; t += blockDim.x) {
            float s = 0.0f;
            for (int w = 0; w < nw; ++w) s += s_acc5[w * N + t];
            part[4 * N + 4 + t] = s;
        }
    if (tid == 0) write_partial_header(P, A, b, chunk, m, Zb);
    publish_and_combine<MATH>(P, A, b, P.blocks_per_ctrl, s_unom, s_red, s_pair, reinterpret_cast<float*>(s_acc), s_vnom);
}

template <int MATH>
__device__ __forceinline__ void block_partial_and_combine(const DevParams& P, const StepArgs& A, const int b,
                                                          const int chunk, const float J, const float lo, const float hi,
                                                          const float4* s_unom, float* s_red, float4* s_acc, float* s_pair,
                                                          const float* s_vnom = nullptr, float* s_acc5 = nullptr,
                                                          const bool stored = false)
{
    const float Jv[1] = {J};
    block_partial_and_combine_n<MATH, 1>(P, A, b, chunk, (uint32_t)(chunk * blockDim.x), Jv, lo, hi, stored, s_unom, s_red,
                                         s_acc, s_pair, s_vnom, s_acc5);
}

// Fused softmax update, second half ("last block done").  Every block of controller b has written
// its partial  part = { S[4N] = sum_k e_k dU_k, m = min_k J_k, Z = sum_k e_k }  with
// e_k = exp(-(J_k - m)/lambda)  (online-softmax form of eq.(4),(5)).  The block that
// takes the last ticket rescales the nb partials to the global minimum beta and writes
//   u_new = u_nom + sum_q S_q exp(-(m_q - beta)/lambda) / Z_tot,   w_k = exp(-(J_k - beta)/lambda) / Z_tot.
// Partials whose rescale factor underflows to 0 contribute exactly 0 and are not read.
//
// This runs after the last rollout of the controller has finished, so it is on the critical path of the
// iteration latency.  Measured with clock64 stamps (profiles/README_r02c.md): round 1's form -- block-wide min,
// sum and compaction, seven __syncthreads -- took 7600 cycles in the block that runs it (5400 with a warm
// instruction cache), of which only ~1500 are the two L2 round trips it needs.  For up to kCombineFast x 32
// partials every WARP therefore derives beta, Z and the list of contributing partials on its own, from registers
// and shuffles (all warps compute the same values in the same order, so the result does not depend on the warp),
// and goes straight on to its columns of u_new and its share of the weights: ticket; (m, Z) pairs together with
// the first costs; S rows of the partials that count -- and no block barrier after the ticket.
// s_pair: 3 nb floats of shared memory.  All threads of the block must call this.
__device__ __forceinline__ unsigned ticket_acq_rel(unsigned* ctr)
{
    unsigned old;
    asm volatile("atom.add.acq_rel.gpu.global.u32 %0, [%1], 1;" : "=r"(old) : "l"(ctr) : "memory");
    return old;
}

constexpr int kCombineFast = 8;        // (m, Z) pairs a lane keeps in registers: per-warp combine for nb <= 256

template <int MATH, int ROWS>
__device__ __forceinline__ void publish_and_combine(const DevParams& P, const StepArgs& A, int b, int nb,
                                                    const float4* s_unom, float* s_red, float* s_pair, float* s_work,
                                                    const float* s_vnom)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, N = P.N, stride = P.part_stride, nthr = blockDim.x;
    const int nw = nthr >> 5;
    int* s_flag = reinterpret_cast<int*>(s_red) + 48;
    int* s_cnt = s_flag + 1;
    __syncthreads();                               // the block's partial is written (CTA-scope order) ...
    if (tid == 0) *s_flag = (ticket_acq_rel(&A.counters[b]) == (unsigned)(nb - 1));   // ... and released here
    if (tid == 0) MPPI_STAMP(A, 8);
    __syncthreads();
    if (!*s_flag) return;
    if (tid == 0) MPPI_STAMP(A, 13);

    const float* pb = A.partials + (size_t)b * nb * stride;
    const float2* hb = A.headers + (size_t)b * nb;
    float* s_scale = s_pair;
    int* s_list = reinterpret_cast<int*>(s_pair + 2 * nb);
    // this thread's first costs (for the weights) go out together with the (m, Z) pairs
    const float4* c4 = reinterpret_cast<const float4*>(A.cost + (size_t)b * P.K);
    const int n4 = P.K >> 2;
    constexpr int PRE = 4;
    float4 cpre[PRE];
#pragma unroll
    for (int r = 0; r < PRE; ++r)
        cpre[r] = tid + r * nthr < n4 ? __ldcg(c4 + tid + r * nthr) : make_float4(0.f, 0.f, 0.f, 0.f);
    const float inf = __int_as_float(0x7f800000);
    float beta, invZ;
    int cnt;
    if (nb <= 32 * kCombineFast) {
        // ---- per warp: registers and shuffles, no block barrier.  The headers are contiguous (8 bytes per partial),
        // so a warp reads all of them in nb / 16 cache lines ----
        float mq[kCombineFast], zq[kCombineFast];
        float bm = inf;
#pragma unroll
        for (int r = 0; r < kCombineFast; ++r) {
            const int j = lane + 32 * r;
            mq[r] = inf; zq[r] = 0.0f;
            if (j < nb) {
                const float2 mz = __ldcg(hb + j);
                mq[r] = mz.x; zq[r] = mz.y;
            }
        }
#pragma unroll
        for (int r = 0; r < kCombineFast; ++r) bm = fminf(bm, mq[r]);
        if (tid == 0) MPPI_STAMP(A, 9);
        beta = warp_min(bm);
        if (tid == 0) MPPI_STAMP(A, 14);
        float zz = 0.0f;
        cnt = 0;
#pragma unroll
        for (int r = 0; r < kCombineFast; ++r) {
            if (32 * r < nb) {                         // uniform
                const float sc = lane + 32 * r < nb ? exp_weight<MATH>((beta - mq[r]) * P.inv_lambda) : 0.0f;
                zz = fmaf(zq[r], sc, zz);
                const bool on = sc != 0.0f;
                const unsigned msk = __ballot_sync(kFull, on);
                if (on) {                              // ascending partial index: deterministic order of the sums
                    const int at = cnt + __popc(msk & ((1u << lane) - 1u));
                    s_list[at] = lane + 32 * r; s_scale[at] = sc;
                }
                cnt += __popc(msk);
            }
        }
        if (tid == 0) MPPI_STAMP(A, 15);
        invZ = 1.0f / warp_sum(zz);                    // fixed butterfly order: identical in every warp
        __syncwarp();                                  // this warp's (identical) copy of the list is visible to its lanes
    } else {
        // ---- general form: block-wide reductions through shared memory ----
        float* s_z = s_pair + nb;
        float bm = inf;
        for (int j = tid; j < nb; j += nthr) {
            const float2 mz = __ldcg(hb + j);
            s_scale[j] = mz.x; s_z[j] = mz.y;
            bm = fminf(bm, mz.x);
        }
        beta = block_min(bm, s_red);
        float zz = 0.0f;
        for (int j = tid; j < nb; j += nthr) {
            const float sc = exp_weight<MATH>((beta - s_scale[j]) * P.inv_lambda);
            zz = fmaf(s_z[j], sc, zz);
            s_scale[j] = sc;
        }
        invZ = 1.0f / block_sum(zz, s_red);      // its barriers also order the s_scale writes
        // deterministic compaction of the partials with a non-zero scale (warp 0, ascending index): (index, scale)
        // pairs; the compacted scales go to s_z, which nobody reads any more
        if (tid < 32) {
            int c = 0;
            for (int j0 = 0; j0 < nb; j0 += 32) {
                const int j = j0 + lane;
                const float sc = j < nb ? s_scale[j] : 0.0f;
                const bool on = sc != 0.0f;
                const unsigned msk = __ballot_sync(kFull, on);
                if (on) { const int at = c + __popc(msk & ((1u << lane) - 1u)); s_list[at] = j; s_z[at] = sc; }
                c += __popc(msk);
            }
            if (lane == 0) *s_cnt = c;
        }
        __syncthreads();
        cnt = *s_cnt;
        s_scale = s_z;
    }
    if (tid == 0) MPPI_STAMP(A, 10);
#ifdef MPPI_TIMELINE
    if (tid == 0) A.timeline[(size_t)(blockIdx.y * gridDim.x + blockIdx.x) * 16 + 3] = (unsigned long long)cnt;
#endif
    // ---- S rows of the contributing partials.  Warp w takes the partials list[w], list[w + nw], ...; its lanes take
    // the columns lane, lane + 32, ... -- every load of the block is in flight at once (one L2 round trip whatever the
    // number of contributing partials; thread-per-column with four loads per round took cnt / 4 round trips).  The
    // warps' sums meet in s_work [nw][group columns] and are added in warp order: deterministic.
    // Column groups: the 4N thrust columns, then (fifth input) the N columns kept after the header.
    // The first batch of loads goes out BEFORE the weights are formed and is consumed after them: the weights need
    // beta and Z only, so their arithmetic and stores fill the L2 round trip of the S rows.
    constexpr int CMAX = 8;                            // columns per lane and sweep: 256 columns per sweep
    constexpr int kRows = ROWS;                        // partials per warp and batch, all loads issued before the first
                                                       // use (4 in the latency kernels, 2 where registers are the rollout's)
    auto load_batch = [&](const int goff, const int gcol, const int c0, const int i0, float (&v)[kRows][CMAX], float (&sc)[kRows]) {
#pragma unroll
        for (int rr = 0; rr < kRows; ++rr) {
            const int i = i0 + rr * nw;
            const bool on = i < cnt;
            sc[rr] = on ? s_scale[i] : 0.0f;
            const float* row = pb + (size_t)(on ? s_list[i] : 0) * stride + goff + c0 + lane;
#pragma unroll
            for (int c = 0; c < CMAX; ++c)
                v[rr][c] = (on && c0 + 32 * c + lane < gcol) ? __ldcg(row + 32 * c) : 0.0f;
        }
    };
    float v0[kRows][CMAX], sc0[kRows];
    load_batch(0, 4 * N, 0, warp, v0, sc0);

    // ---- weights w_k = exp(-(J_k - beta) / lambda) / Z ----
    float4* w4 = reinterpret_cast<float4*>(A.weights + (size_t)b * P.K);
    const float nil = -P.inv_lambda;
    int nz = 0;                                // samples of this thread that carry weight
    auto weights_of = [&](const float4 c) {
        const float4 w = make_float4(exp_weight<MATH>((c.x - beta) * nil) * invZ, exp_weight<MATH>((c.y - beta) * nil) * invZ,
                                     exp_weight<MATH>((c.z - beta) * nil) * invZ, exp_weight<MATH>((c.w - beta) * nil) * invZ);
        nz += (w.x > 0.0f) + (w.y > 0.0f) + (w.z > 0.0f) + (w.w > 0.0f);
        return w;
    };
#pragma unroll
    for (int r = 0; r < PRE; ++r) {
        const int i = tid + r * nthr;
        if (i < n4) w4[i] = weights_of(cpre[r]);
    }
#pragma unroll 4
    for (int i = tid + PRE * nthr; i < n4; i += nthr) w4[i] = weights_of(__ldcg(c4 + i));
    if (tid == 0) MPPI_STAMP(A, 11);

    const float* unf = reinterpret_cast<const float*>(s_unom);
    for (int grp = 0; grp < (s_vnom ? 2 : 1); ++grp) {
        const int gcol = grp ? N : 4 * N, goff = grp ? 4 * N + 4 : 0;
        for (int c0 = 0; c0 < gcol; c0 += 32 * CMAX) {
            float acc[CMAX];
#pragma unroll
            for (int c = 0; c < CMAX; ++c) acc[c] = 0.0f;
            for (int i0 = warp; i0 < cnt; i0 += kRows * nw) {
                float v[kRows][CMAX], sc[kRows];
                if (grp == 0 && c0 == 0 && i0 == warp) {           // the batch that is already in registers
#pragma unroll
                    for (int rr = 0; rr < kRows; ++rr) {
                        sc[rr] = sc0[rr];
#pragma unroll
                        for (int c = 0; c < CMAX; ++c) v[rr][c] = v0[rr][c];
                    }
                } else {
                    load_batch(goff, gcol, c0, i0, v, sc);
                }
#pragma unroll
                for (int rr = 0; rr < kRows; ++rr)
#pragma unroll
                    for (int c = 0; c < CMAX; ++c) acc[c] = fmaf(v[rr][c], sc[rr], acc[c]);
            }
#pragma unroll
            for (int c = 0; c < CMAX; ++c)
                if (c0 + 32 * c + lane < gcol) s_work[warp * gcol + c0 + 32 * c + lane] = acc[c];
        }
        __syncthreads();
        for (int j = tid; j < gcol; j += nthr) {
            float s = 0.0f;
            for (int w = 0; w < nw; ++w) s += s_work[w * gcol + j];
            if (grp == 0) A.u_new[(size_t)b * 4 * N + j] = fmaf(s, invZ, unf[j]);
            else A.v_new[(size_t)b * N + j] = fmaf(s, invZ, s_vnom[j]);
        }
        if (s_vnom) __syncthreads();                   // s_work is reused by the next group
    }
    if (A.hint) {
        // Hint for the NEXT launch on this controller (keeps_du): did many samples carry weight?  Then the sparse
        // re-derivation of the block partials costs a second pass over the noise stream and storing dU is cheaper.
        const float nnz = block_sum((float)nz, s_red);
        if (tid == 0) A.hint[b] = nnz * 32.0f > (float)P.K ? 1u : 0u;
    }
    if (tid == 0) A.counters[b] = 0u;          // ready for the next launch
    if (A.done_flag) {
        // host-polled completion: every output store of this block is made visible system-wide, then
        // the block that finishes the last controller raises the flag in mapped host memory
        __threadfence_system();
        __syncthreads();
        if (tid == 0) {
            bool all = true;
            if (P.B > 1) {
                all = atomicAdd(&A.counters[P.B], 1u) == (unsigned)(P.B - 1);
                if (all) A.counters[P.B] = 0u;
                __threadfence_system();
            }
            if (all) *reinterpret_cast<volatile unsigned*>(A.done_flag) = A.done_value;
        }
    }
}

}  // namespace mppi
