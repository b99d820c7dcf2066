// mppi_static.cu -- mppi_step_static: one MPPI iteration that allocates NOTHING.
//
// For callers that cannot call cudaMalloc -- code under CUDA-graph capture, tight serving loops, harnesses that forbid
// it.  The existing path (mppi_create + mppi_set_gates + mppi_step) allocates its scratch (block partials, (m, Z)
// headers, tickets) and the packed gate table with cudaMalloc.  This entry point runs the SAME iteration -- gate
// progress (MPPI_OBJ_GATE), rotor-thrust inputs, fused pipeline, the pipelined latency kernel
// rollout_pipe_kernel<OBJ_GATE> -- with all of that in ONE file-scope `static __device__` array of a stated maximum
// size: MPPI_STATIC_MAX_K samples, MPPI_STATIC_MAX_N steps, MPPI_STATIC_MAX_B controllers, MPPI_STATIC_MAX_GATES
// gates, ~1.07 MB that every GPU which loads the library holds until the process exits.
//
// It calls no cudaMalloc / cudaFree / cudaHostAlloc and no allocating library routine; the caller passes every input
// and output as a device pointer.  In host code the array's name is only a host-side stand-in, not a device address:
// the device address is taken once per device with cudaGetSymbolAddress (checked) and handed to the kernels; the small
// set-up kernel of this file names the array directly.
//
// Every call shares the array, which keeps the last call's contents.  What must start at zero (the last-block
// tickets) is cleared by every call.  Calls that overlap on the GPU -- two streams, two host threads, two graphs
// replayed concurrently -- race on it and give wrong results: keep the calls of one device stream-ordered.
#include <cstdio>
#include <cstring>
#include <cmath>
#include <mutex>

#include "../../include/mppi.h"
#include "mppi_internal.h"
#include "mppi_rollout.cuh"
#include "mppi_pipe.cuh"

using namespace mppi;

namespace {

// ---- layout of the static scratch (units: floats; every region starts on a 256-byte boundary) ----------------------
constexpr int kMaxBlocks = MPPI_STATIC_MAX_K / 32;                               // pipelined kernel: 32 samples per block
constexpr int kMaxStride = (4 * MPPI_STATIC_MAX_N + 4 + 7) & ~7;                 // floats per partial (as mppi_create)
constexpr size_t kOffPartials = 0;
constexpr size_t kNumPartials = (size_t)MPPI_STATIC_MAX_B * kMaxBlocks * kMaxStride;
constexpr size_t kOffHeaders = kOffPartials + kNumPartials;                      // float2 per partial
constexpr size_t kNumHeaders = (size_t)MPPI_STATIC_MAX_B * kMaxBlocks * 2;
constexpr size_t kOffGates = kOffHeaders + kNumHeaders;                          // [G][4] float4
constexpr size_t kNumGates = (size_t)MPPI_STATIC_MAX_GATES * 16;
constexpr size_t kOffCounters = kOffGates + kNumGates;                           // [B + 1] unsigned, padded
constexpr size_t kNumCounters = 64;
constexpr size_t kScratchFloats = kOffCounters + kNumCounters;
static_assert(kOffHeaders % 64 == 0 && kOffGates % 64 == 0 && kOffCounters % 64 == 0, "regions are 256-byte aligned");

static __device__ __align__(256) float g_static_scratch[kScratchFloats];        // ~1.07 MB per GPU, held until exit

// Set-up kernel of every call (one block): packs the caller's gates [G][11] into the float4 layout the rollout kernels
// read -- (c, a_h) (n, a_v) (h, n.c) (v = h x n, 0), the plane offset and the cross product in double WITHOUT fused
// multiply-adds, i.e. the arithmetic of mppi_set_gates on the host -- and clears the tickets.  Names the array directly.
__global__ void static_setup_kernel(const float* __restrict__ gates, const int G, const int B)
{
    const int i = threadIdx.x;
    if (i < G) {
        const float* r = gates + 11 * i;
        const double c0 = r[0], c1 = r[1], c2 = r[2], n0 = r[3], n1 = r[4], n2 = r[5], h0 = r[6], h1 = r[7], h2 = r[8];
        const double vx = __dsub_rn(__dmul_rn(h1, n2), __dmul_rn(h2, n1));
        const double vy = __dsub_rn(__dmul_rn(h2, n0), __dmul_rn(h0, n2));
        const double vz = __dsub_rn(__dmul_rn(h0, n1), __dmul_rn(h1, n0));
        const double nc = __dadd_rn(__dadd_rn(__dmul_rn(n0, c0), __dmul_rn(n1, c1)), __dmul_rn(n2, c2));
        float4* g = reinterpret_cast<float4*>(g_static_scratch + kOffGates) + 4 * i;
        g[0] = make_float4(r[0], r[1], r[2], r[9]);
        g[1] = make_float4(r[3], r[4], r[5], r[10]);
        g[2] = make_float4(r[6], r[7], r[8], (float)nc);
        g[3] = make_float4((float)vx, (float)vy, (float)vz, 0.0f);
    }
    if (i <= B) reinterpret_cast<unsigned*>(g_static_scratch + kOffCounters)[i] = 0u;
}

// ---- per-device set-up, once: the array's device address and the kernels' shared-memory limit ----------------------
constexpr int kMaxDevices = 64;
std::mutex g_mu;
float* g_dev_ptr[kMaxDevices] = {};
bool g_dev_ready[kMaxDevices] = {};

thread_local char g_err[256] = "";

int fail(int code, const char* fmt, long a = 0, long b = 0)
{
    std::snprintf(g_err, sizeof g_err, fmt, a, b);
    return code;
}

size_t pipe_smem(const DevParams& P)
{
    LaunchCfg c;
    std::memset(&c, 0, sizeof c);
    c.objective = OBJ_GATE; c.fused = 1; c.pipe = 1; c.block_threads = kPipeThreads;
    return rollout_smem_bytes(P, c);
}

}  // namespace

extern "C" const char* mppi_step_static_error(void) { return g_err; }

extern "C" int mppi_step_static(const mppi_params* p, const float* d_gates, int G, const float* d_x0, const int32_t* d_start,
                                const float* d_u_nom, uint64_t seed, uint32_t iter, float* d_u_new, float* d_cost,
                                float* d_weights, void* stream)
{
    if (!p || !d_gates || !d_x0 || !d_start || !d_u_nom || !d_u_new || !d_cost || !d_weights)
        return fail(MPPI_E_NULL, "mppi_step_static: NULL argument");
    if (p->struct_size != sizeof(mppi_params)) return fail(MPPI_E_PARAM, "mppi_step_static: struct_size does not match this library");
    // ---- the limits of the static scratch ----
    if (p->K <= 0 || p->K % 32 != 0) return fail(MPPI_E_PARAM, "mppi_step_static: K must be a positive multiple of 32");
    if (p->K > MPPI_STATIC_MAX_K) return fail(MPPI_E_RANGE, "mppi_step_static: K = %ld exceeds MPPI_STATIC_MAX_K = %ld", p->K, MPPI_STATIC_MAX_K);
    if (p->N < 1) return fail(MPPI_E_PARAM, "mppi_step_static: N must be >= 1");
    if (p->N > MPPI_STATIC_MAX_N) return fail(MPPI_E_RANGE, "mppi_step_static: N = %ld exceeds MPPI_STATIC_MAX_N = %ld", p->N, MPPI_STATIC_MAX_N);
    if (p->B < 1) return fail(MPPI_E_PARAM, "mppi_step_static: B must be >= 1");
    if (p->B > MPPI_STATIC_MAX_B) return fail(MPPI_E_RANGE, "mppi_step_static: B = %ld exceeds MPPI_STATIC_MAX_B = %ld", p->B, MPPI_STATIC_MAX_B);
    if (G < 1 || G > MPPI_STATIC_MAX_GATES) return fail(MPPI_E_RANGE, "mppi_step_static: G = %ld is outside 1..MPPI_STATIC_MAX_GATES = %ld", G, MPPI_STATIC_MAX_GATES);
    // ---- the one configuration this entry point runs ----
    if (p->objective != MPPI_OBJ_GATE || p->input_model != 0 || p->pipeline != MPPI_PIPE_FUSED || p->store_noise != 0 ||
        p->block_threads != 0 || (p->variant != MPPI_VARIANT_AUTO && p->variant != MPPI_VARIANT_PIPELINED))
        return fail(MPPI_E_PARAM, "mppi_step_static: gate objective, rotor-thrust inputs, fused pipeline, no stored noise, block_threads 0, variant AUTO or PIPELINED only");
    auto pos = [](float v) { return std::isfinite(v) && v > 0.0f; };
    if (!pos(p->dt) || !pos(p->lambda) || !pos(p->mass) || !pos(p->Jx) || !pos(p->Jy) || !pos(p->Jz) ||
        !(std::isfinite(p->sigma) && p->sigma >= 0.0f) || !(std::isfinite(p->T_min) && std::isfinite(p->T_max) && p->T_min <= p->T_max) ||
        !std::isfinite(p->arm) || !std::isfinite(p->c_tau) || !std::isfinite(p->g))
        return fail(MPPI_E_PARAM, "mppi_step_static: dt, lambda, mass, inertia > 0; sigma >= 0; T_min <= T_max; arm, c_tau, g finite");
    if (p->drag_x != 0.0f || p->drag_y != 0.0f || p->drag_z != 0.0f || p->w_limit != 0.0f)
        return fail(MPPI_E_PARAM, "mppi_step_static: rotor drag and the body-rate limit cost need input_model = 1 (not available here)");
    const size_t ub = (size_t)p->B * p->N * 4 * sizeof(float);
    {
        const char* x = (const char*)d_u_new; const char* y = (const char*)d_u_nom;
        if (x != y && x < y + ub && y < x + ub) return fail(MPPI_E_RANGE, "mppi_step_static: d_u_new partially overlaps d_u_nom");
    }

    // ---- once per device, with that device current: the array's device address, the kernels' shared-memory limit ----
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(MPPI_E_CUDA, "mppi_step_static: no CUDA device");
    if (dev < 0 || dev >= kMaxDevices) return fail(MPPI_E_RANGE, "mppi_step_static: device ordinal %ld beyond %ld", dev, kMaxDevices - 1);
    float* scratch = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_mu);
        if (!g_dev_ready[dev]) {
            float* ptr = nullptr;
            e = cudaGetSymbolAddress((void**)&ptr, g_static_scratch);
            if (e != cudaSuccess || !ptr) return fail(MPPI_E_CUDA, "mppi_step_static: cudaGetSymbolAddress failed (%ld)", (long)e);
            DevParams worst;
            std::memset(&worst, 0, sizeof worst);
            worst.N = MPPI_STATIC_MAX_N; worst.G = MPPI_STATIC_MAX_GATES; worst.blocks_per_ctrl = kMaxBlocks;
            const int smem_max = (int)pipe_smem(worst);
            e = cudaFuncSetAttribute(rollout_pipe_kernel<OBJ_GATE, 0, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max);
            if (e == cudaSuccess)
                e = cudaFuncSetAttribute(rollout_pipe_kernel<OBJ_GATE, 1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max);
            if (e != cudaSuccess) return fail(MPPI_E_CUDA, "mppi_step_static: cudaFuncSetAttribute failed (%ld)", (long)e);
            g_dev_ptr[dev] = ptr;
            g_dev_ready[dev] = true;
        }
        scratch = g_dev_ptr[dev];
    }

    // ---- derived constants: as mppi_create computes them (in double from the fp32 parameters, rounded once) ----
    DevParams d;
    std::memset(&d, 0, sizeof d);
    d.K = p->K; d.N = p->N; d.B = p->B; d.window = p->window; d.G = G;
    {
        const double h = (double)p->dt;
        d.h2 = (float)(h / 2); d.h3 = (float)(h / 3); d.h4 = (float)(h / 4); d.h6 = (float)(h / 6);
        d.h12 = (float)(h / 12); d.hh2 = (float)(h * h / 2); d.hh3 = (float)(h * h / 3);
    }
    d.dt = p->dt; d.inv_lambda = (float)(1.0 / (double)p->lambda); d.sigma = p->sigma;
    d.bm_k = (float)(-2.0 * 0.6931471805599453 * (double)p->sigma * (double)p->sigma);
    d.T_min = p->T_min; d.T_max = p->T_max;
    d.inv_mass = (float)(1.0 / (double)p->mass); d.g = p->g;
    d.hover = (float)((double)p->mass * (double)p->g / 4.0);
    const double lever = (double)p->arm / std::sqrt(2.0);
    d.ltx = (float)(lever / p->Jx); d.lty = (float)(lever / p->Jy); d.ltz = (float)((double)p->c_tau / p->Jz);
    d.gyx = (float)(((double)p->Jy - p->Jz) / p->Jx);
    d.gyy = (float)(((double)p->Jz - p->Jx) / p->Jy);
    d.gyz = (float)(((double)p->Jx - p->Jy) / p->Jz);
    d.w_omega = p->w_omega; d.miss = p->gate_miss_penalty; d.bonus = p->gate_pass_bonus;
    d.blocks_per_ctrl = p->K / 32;
    d.part_stride = (4 * p->N + 4 + 7) & ~7;
    d.pipe_d = 4; d.pipe_df = 3;
    d.gates = reinterpret_cast<const float4*>(scratch + kOffGates);

    StepArgs a;
    std::memset(&a, 0, sizeof a);
    a.x0 = d_x0; a.start = d_start; a.u_nom = d_u_nom; a.u_new = d_u_new; a.cost = d_cost; a.weights = d_weights;
    a.partials = scratch + kOffPartials;
    a.headers = reinterpret_cast<float2*>(scratch + kOffHeaders);
    a.counters = reinterpret_cast<unsigned*>(scratch + kOffCounters);
    a.seed_lo = (uint32_t)(seed & 0xffffffffu); a.seed_hi = (uint32_t)(seed >> 32); a.iter = iter;
    for (uint32_t r = 0; r < 10; ++r) {          // Philox key schedule (Weyl sequence)
        a.rk[2 * r] = a.seed_lo + r * 0x9E3779B9u;
        a.rk[2 * r + 1] = a.seed_hi + r * 0xBB67AE85u;
    }

    const size_t smem = pipe_smem(d);
    cudaStream_t s = (cudaStream_t)stream;
    static_setup_kernel<<<1, 64, 0, s>>>(d_gates, G, p->B);
    const dim3 grid(d.blocks_per_ctrl, d.B), block(kPipeThreads);
    if (p->fast_math) rollout_pipe_kernel<OBJ_GATE, 1, false><<<grid, block, smem, s>>>(d, a);
    else rollout_pipe_kernel<OBJ_GATE, 0, false><<<grid, block, smem, s>>>(d, a);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(MPPI_E_CUDA, "mppi_step_static: kernel launch failed (%ld)", (long)e);
    g_err[0] = 0;
    return MPPI_OK;
}
