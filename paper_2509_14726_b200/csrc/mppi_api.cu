// mppi_api.cu -- host side of libmppi: the C ABI declared in include/mppi.h.
// Parameter validation, track packing, scratch allocation, stream launches and CUDA-graph replay.
#include <algorithm>
#include <atomic>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/mppi.h"
#include "mppi_cost.cuh"
#include "mppi_internal.h"

using namespace mppi;

struct GraphSlot {
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    std::vector<cudaGraphNode_t> rollout_nodes, reduce_nodes;
    int n_iters = 0;
};

struct mppi_ctx {
    mppi_params prm;
    DevParams dp;
    LaunchCfg cfg;
    int device = 0, sm_count = 0, l2_bytes = 0;
    int lazy_pipe = 0, scalar_tpb = 0, scalar_packed = 0;     // input_model = 1: pipelined kernel iff it fits in shared memory (decided in prepare)
    bool have_gates = false, have_ref = false, have_path = false;
    float4* d_gates = nullptr;
    float4* d_ref = nullptr;
    float4* d_path = nullptr;
    float4* d_du = nullptr;
    float* d_partials = nullptr;
    float2* d_headers = nullptr;
    unsigned* d_counters = nullptr;
    unsigned* d_hint = nullptr;            // [B] dense-weights hint of the previous iteration (StepArgs::hint)
    bool keep_du = false;                  // d_du belongs to the caller-visible contract (two-pass / store_noise)
    bool du_tried = false;
    const int* d_prev_front = nullptr;     // caller-owned (mppi_set_prev_front)
    const float* d_v_nom = nullptr; float* d_v_new = nullptr;   // caller-owned (mppi_set_progress)
    // device staging for mppi_step_host
    float* d_hx0 = nullptr; int* d_hstart = nullptr; float* d_hu = nullptr; float* d_hcost = nullptr;
    float* d_hw = nullptr;
    // mapped pinned host staging of mppi_step_host: the inputs go down in ONE packed copy (reading them
    // from host memory inside the kernel costs thousands of small bus reads -- measured slower), the
    // kernel writes its outputs straight into host memory and raises a flag the host polls
    unsigned char* h_pin = nullptr; unsigned char* d_pin = nullptr; unsigned char* d_in = nullptr;
    size_t pin_x0 = 0, pin_start = 0, pin_u = 0, pin_unew = 0, pin_cost = 0, pin_w = 0, pin_flag = 0, pin_bytes = 0;
    unsigned host_seq = 0;
    int xdim = 13;         // floats per state row: 13, or 17 under the thrust-rate input model
    int64_t scratch_bytes = 0;
    int64_t launches = 0;
    GraphSlot g_step, g_opt;
    std::string err;
};

static thread_local std::string g_create_err;

static int fail(mppi_ctx* c, int code, const std::string& msg)
{
    if (c) c->err = msg; else g_create_err = msg;
    return code;
}
static int cuda_fail(mppi_ctx* c, cudaError_t e, const char* what)
{
    return fail(c, MPPI_E_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
#define CK(ctx, call)                                              \
    do {                                                           \
        cudaError_t e_ = (call);                                   \
        if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call);   \
    } while (0)

extern "C" const char* mppi_error_string(int s)
{
    switch (s) {
        case MPPI_OK: return "ok";
        case MPPI_E_NULL: return "null pointer";
        case MPPI_E_PARAM: return "parameter out of range";
        case MPPI_E_NO_TRACK: return "track data for this objective not set";
        case MPPI_E_TRACK: return "track data rejected";
        case MPPI_E_RANGE: return "buffer overlap or count out of range";
        case MPPI_E_CUDA: return "CUDA error";
        case MPPI_E_ALLOC: return "allocation failed";
        default: return "unknown status";
    }
}

extern "C" const char* mppi_last_error(mppi_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

extern "C" int mppi_default_params(mppi_params* p)
{
    if (!p) return fail(nullptr, MPPI_E_NULL, "mppi_default_params: p is NULL");
    std::memset(p, 0, sizeof *p);
    p->struct_size = sizeof *p;
    p->K = 256; p->N = 20; p->B = 1; p->objective = MPPI_OBJ_GATE;
    p->dt = 0.02f; p->lambda = 1.0f; p->sigma = 1.0f;
    p->mass = 0.85f; p->Jx = 1e-3f; p->Jy = 1e-3f; p->Jz = 1.7e-3f;
    p->arm = 0.15f; p->c_tau = 0.016f; p->g = 9.81f;
    p->T_min = 0.0f; p->T_max = 7.0f;
    p->w_omega = 0.01f; p->gate_miss_penalty = 10.0f; p->gate_pass_bonus = 5.0f;
    p->Qp = 100.0f; p->Qv = 1.0f; p->Qq = 10.0f; p->Qw = 0.1f; p->R = 0.01f;
    p->q_contour = 200.0f; p->q_lag = 50.0f; p->mu_progress = 2.0f;
    p->window = 16;
    p->pipeline = MPPI_PIPE_FUSED; p->use_graph = 0; p->block_threads = 0; p->fast_math = 0;
    p->store_noise = 0; p->variant = MPPI_VARIANT_AUTO;
    p->q_near = 0.0f; p->r_near = 0.0f;
    p->input_model = 0; p->rate_max = 0.0f; p->drag_x = p->drag_y = p->drag_z = 0.0f;
    p->w_limit = 0.0f; p->omega_max = 0.0f;
    p->sigma_v = 0.0f; p->dv_max = 0.0f; p->v_theta_max = 0.0f; p->r_dv = 0.0f;
    p->near_mode = 0;
    return MPPI_OK;
}

static bool finite_pos(float v) { return std::isfinite(v) && v > 0.0f; }

// May the time-parallel kernel (mppi_scan.cuh) run this configuration?  Its body-rate scan needs the equations of
// omega_x, omega_y to be linear given omega_z: Jx == Jy (then (Jx - Jy)/Jz = 0 and (Jy - Jz)/Jx = -(Jz - Jx)/Jy).
static bool scan_capable(const mppi_params* p)
{
    return p->input_model == 0 && (p->objective == MPPI_OBJ_GATE || p->objective == MPPI_OBJ_GATE_PAPER) && p->Jx == p->Jy && p->N <= 64 &&
           p->pipeline == MPPI_PIPE_FUSED && p->block_threads == 0 && p->K % 32 == 0;
}
// Samples per block of the time-parallel kernel (16 lanes each): 32, or fewer (even, >= 8) when that lets the blocks
// of the B controllers cover every SM -- its blocks run one per SM.  configs[1] on 148 SMs: 28 -> 147 blocks.
static int scan_samples_per_block(const mppi_params* p, int sm_count)
{
    int64_t nb = p->K / 32;
    const int64_t room = sm_count / p->B;            // blocks per controller that still fit in one wave
    if (room > nb) nb = std::min<int64_t>(room, p->K / 8);
    const int spb = 2 * (int)((p->K + 2 * nb - 1) / (2 * nb));
    return std::min(32, std::max(8, spb));
}

static int validate(const mppi_params* p)
{
#define BAD(cond, msg) if (cond) return fail(nullptr, MPPI_E_PARAM, msg)
    BAD(p->struct_size != sizeof(mppi_params), "struct_size does not match this library");
    BAD(p->K <= 0 || p->K % 32 != 0, "K must be a positive multiple of 32");
    BAD(p->N <= 0 || p->N > MPPI_MAX_N, "N must be in 1..MPPI_MAX_N");
    BAD(p->B <= 0 || p->B > 65535, "B must be in 1..65535");
    BAD(p->objective < 0 || p->objective > 4, "objective must be 0..4");
    if (p->objective == MPPI_OBJ_CONTOUR_PAPER) {
        BAD(p->input_model != 1, "MPPI_OBJ_CONTOUR_PAPER needs input_model = 1 (its inputs are thrust rates)");
        BAD(p->pipeline != MPPI_PIPE_FUSED || p->use_graph, "MPPI_OBJ_CONTOUR_PAPER: fused pipeline, no graph replay");
        BAD(!(std::isfinite(p->sigma_v) && p->sigma_v >= 0.0f) || !(p->dv_max > 0.0f) || !(p->v_theta_max > 0.0f) ||
                !(std::isfinite(p->r_dv) && p->r_dv >= 0.0f), "need sigma_v >= 0, dv_max > 0, v_theta_max > 0, r_dv >= 0");
    }
    BAD(!(std::isfinite(p->q_near) && p->q_near >= 0.0f) || !(std::isfinite(p->r_near) && p->r_near >= 0.0f),
        "q_near and r_near must be >= 0");
    BAD(p->near_mode != 0 && p->near_mode != 1, "near_mode must be 0 or 1");
    BAD(!finite_pos(p->dt), "dt must be > 0");
    BAD(!finite_pos(p->lambda), "lambda must be > 0");
    BAD(!(std::isfinite(p->sigma) && p->sigma >= 0.0f), "sigma must be >= 0");
    BAD(!finite_pos(p->mass) || !finite_pos(p->Jx) || !finite_pos(p->Jy) || !finite_pos(p->Jz),
        "mass and inertia must be > 0");
    BAD(!std::isfinite(p->arm) || !std::isfinite(p->c_tau) || !std::isfinite(p->g), "arm, c_tau, g must be finite");
    BAD(!(std::isfinite(p->T_min) && std::isfinite(p->T_max) && p->T_min <= p->T_max), "need T_min <= T_max");
    BAD(p->window < 1 || p->window > MPPI_MAX_WINDOW, "window must be in 1..MPPI_MAX_WINDOW");
    BAD(p->pipeline != MPPI_PIPE_FUSED && p->pipeline != MPPI_PIPE_TWO_PASS, "unknown pipeline");
    BAD(p->block_threads != 0 && (p->block_threads < 32 || p->block_threads > 256 || p->block_threads % 32 != 0 ||
                                  p->K % p->block_threads != 0),
        "block_threads must be 0 or a multiple of 32 in 32..256 that divides K");
    BAD((int64_t)p->K / 32 > 65535, "K too large");
    BAD(p->variant < 0 || p->variant > 5, "unknown variant");
    BAD(p->variant == MPPI_VARIANT_SCAN && !scan_capable(p),
        "the time-parallel variant needs input_model 0, objective MPPI_OBJ_GATE or MPPI_OBJ_GATE_PAPER, Jx == Jy, N <= 64, the fused pipeline, "
        "block_threads 0");
    BAD(p->variant == MPPI_VARIANT_PACKED &&
            (p->K % 64 != 0 || (p->block_threads && (p->block_threads > 128 || p->K % (2 * p->block_threads) != 0))),
        "the packed variant needs K % 64 == 0, block_threads <= 128 and 2*block_threads dividing K");
    BAD((p->variant == MPPI_VARIANT_LATENCY || p->variant == MPPI_VARIANT_PIPELINED) && p->pipeline != MPPI_PIPE_FUSED,
        "the latency variants need the fused pipeline");
    BAD(p->input_model != 0 && p->input_model != 1, "input_model must be 0 or 1");
    auto nonneg = [](float v) { return std::isfinite(v) && v >= 0.0f; };
    BAD(!nonneg(p->drag_x) || !nonneg(p->drag_y) || !nonneg(p->drag_z) || !nonneg(p->w_limit) || !nonneg(p->omega_max) ||
            !nonneg(p->rate_max), "drag, w_limit, omega_max, rate_max must be >= 0");
    if (p->input_model == 0) {
        BAD(p->drag_x != 0.0f || p->drag_y != 0.0f || p->drag_z != 0.0f || p->w_limit != 0.0f,
            "rotor drag and the body-rate limit cost need input_model = 1");
    } else {
        BAD(!(p->rate_max > 0.0f), "rate_max must be > 0 when input_model = 1");
        BAD(p->variant != MPPI_VARIANT_AUTO && p->variant != MPPI_VARIANT_THROUGHPUT && p->variant != MPPI_VARIANT_PIPELINED &&
                p->variant != MPPI_VARIANT_PACKED,
            "input_model = 1 has scalar and packed throughput kernels and a pipelined latency kernel: variant must not be LATENCY");
        BAD(p->variant == MPPI_VARIANT_PACKED &&
                (p->K % 64 != 0 || p->objective == MPPI_OBJ_CONTOUR),
            "input_model = 1, PACKED: K % 64 == 0, not the search-based contouring");
        BAD(p->variant == MPPI_VARIANT_PIPELINED &&
                (p->pipeline != MPPI_PIPE_FUSED || p->block_threads != 0 || p->N > 100 || p->K % 32 != 0 ||
                 p->objective == MPPI_OBJ_CONTOUR),
            "input_model = 1, PIPELINED: fused pipeline, block_threads 0, N <= 100, K % 32 == 0, not the search-based contouring");
    }
#undef BAD
    return MPPI_OK;
}

// Launch shape.  Latency variant: C rollout warps per 256-thread block, the smallest C in {1,2,4}
// that brings the grid down to one block per SM (so every rollout warp owns a scheduler).
// Throughput variant: 256-thread blocks when the grid still covers the chip several times, else 128.
// input_model = 1: may the pipelined latency kernel (mppi_pipe_rate.cuh) run this configuration at all?
static bool rate_pipe_candidate(const mppi_params* p, int sm_count)
{
    if (p->input_model != 1 || p->pipeline != MPPI_PIPE_FUSED || p->block_threads != 0 || p->N > 100 || p->K % 32 != 0 ||
        p->objective == MPPI_OBJ_CONTOUR || p->use_graph)
        return false;
    if (p->variant == MPPI_VARIANT_PIPELINED) return true;
    return p->variant == MPPI_VARIANT_AUTO && (int64_t)p->B * p->K / 32 <= 2 * (int64_t)sm_count;
}

// AUTO (input_model = 0), from the batch sweep of profiles/sweep_r02*.md (K = 4096, N = 50, B = 1 .. 64; warps = B K / 32):
//   warps <= 2 SMs   pipelined kernel: its 32-sample blocks run two per SM, so this is one wave
//   warps <= 8 SMs   latency kernel with C = 4 rollout warps per block (the pipelined kernel would need several
//                    waves of latency-bound blocks; the throughput kernels cannot fill the chip yet)
//   warps <= 12 SMs  scalar throughput kernel (the packed kernel's grid is half as many blocks: under one wave)
//   above            packed fp32x2 throughput kernel (scalar when K % 64 != 0)
// search-based contouring (objective 2): the window search is 2/3 of a step and cannot be split over the pipeline's
// roles: latency kernel up to 4 SMs warps, scalar throughput kernel up to 12 SMs warps, packed above.
// `avoid` (prepare(), when the preferred kernel does not fit in shared memory with the track that was set):
// bit 0 = not the pipelined kernel, bit 1 = not the latency kernel either.
static void pick_shape(const mppi_params* p, int sm_count, int* block_threads, int* lat_consumers, int* packed, int* pipe,
                       int* scan, int avoid = 0)
{
    const int64_t warps = (int64_t)p->B * p->K / 32;
    *lat_consumers = 0;
    *packed = 0;
    *pipe = 0;
    *scan = 0;
    // time-parallel kernel: on request, or (AUTO) whenever it can run and its blocks fit in one wave of one block
    // per SM -- cfg1: 17.6 us against 18.8 us for the pipelined kernel in its first form (profiles/README_r02f.md)
    if (p->variant == MPPI_VARIANT_SCAN ||          // validate() has checked scan_capable
        (p->variant == MPPI_VARIANT_AUTO && scan_capable(p) && warps <= sm_count && !(avoid & 1))) {
        *scan = scan_samples_per_block(p, sm_count); *block_threads = 16 * *scan;
        return;
    }
    if (p->input_model == 1) {                     // thrust-rate model: its own kernels (mppi_rate.cu)
        // the scalar shape; whether the pipelined latency kernel takes over is decided in prepare(), once the
        // track (and with it the shared-memory footprint) is known -- see rate_pipe_candidate
        // objective 4 runs on the packed kernel too, but no faster than on the scalar one (313 vs 307 us x 64: its
        // two Philox blocks per sample-step, path look-ups and stage costs stay scalar per half): AUTO keeps the scalar
        const bool pk_obj = p->objective != MPPI_OBJ_CONTOUR &&
                            (p->variant == MPPI_VARIANT_PACKED || p->objective != MPPI_OBJ_CONTOUR_PAPER);
        // packed fp32x2 throughput kernel (rollout_rate2_kernel): when the grid covers the chip
        if (pk_obj && p->K % 64 == 0 && (p->variant == MPPI_VARIANT_PACKED ||
                                         (p->variant == MPPI_VARIANT_AUTO && warps >= 8 * (int64_t)sm_count))) {
            if (!p->block_threads || (p->block_threads <= 128 && p->K % (2 * p->block_threads) == 0)) {
                *packed = 1;
                if (p->block_threads) { *block_threads = p->block_threads; return; }
                for (int tpb : {128, 64, 32})
                    if (p->K % (2 * tpb) == 0) { *block_threads = tpb; return; }
            }
        }
        if (p->block_threads) { *block_threads = p->block_threads; return; }
        for (int tpb : {128, 64, 32})
            if (p->K % tpb == 0) { *block_threads = tpb; return; }
    }
    const bool lat_ok = p->pipeline == MPPI_PIPE_FUSED && p->block_threads == 0;
    const bool automatic = p->variant == MPPI_VARIANT_AUTO;
    const bool search = p->objective == MPPI_OBJ_CONTOUR;
    const bool want_pipe = p->variant == MPPI_VARIANT_PIPELINED ||
                           (automatic && !search && warps <= 2 * (int64_t)sm_count && !(avoid & 1));
    if (lat_ok && want_pipe) {
        *pipe = 1; *block_threads = 256;
        return;
    }
    const bool want_lat = p->variant == MPPI_VARIANT_LATENCY ||
                          (automatic && !(avoid & 2) && warps <= (search ? 4 : 8) * (int64_t)sm_count);
    if (lat_ok && want_lat) {
        int best = 0;
        for (int c : {1, 2, 4})
            if (p->K % (32 * c) == 0) {
                best = c;
                if (warps / c <= sm_count) break;
            }
        if (best) { *lat_consumers = best; *block_threads = 256; return; }
    }
    // packed fp32x2 throughput kernel: two samples per thread
    const bool small_grid = automatic && warps <= 12 * (int64_t)sm_count;      // the packed grid (half as many blocks) would not cover the chip
    if (p->K % 64 == 0 && !small_grid &&
        (p->variant == MPPI_VARIANT_PACKED ||
         (automatic && (!p->block_threads || (p->block_threads <= 128 && p->K % (2 * p->block_threads) == 0))))) {
        *packed = 1;
        if (p->block_threads) { *block_threads = p->block_threads; return; }
        for (int tpb : {128, 64, 32})
            if (p->K % (2 * tpb) == 0) { *block_threads = tpb; return; }
    }
    if (p->block_threads) { *block_threads = p->block_threads; return; }
    if (p->K % 256 == 0 && warps >= 16 * (int64_t)sm_count) { *block_threads = 256; return; }
    for (int tpb : {128, 64, 32})
        if (p->K % tpb == 0) { *block_threads = tpb; return; }
    *block_threads = 32;
}

static int blocks_per_ctrl_of(const mppi_params* p, const LaunchCfg& cfg)
{
    return cfg.scan ? (p->K + cfg.scan - 1) / cfg.scan : cfg.pipe ? p->K / 32 : cfg.lat_consumers ? p->K / (32 * cfg.lat_consumers)
                                                    : p->K / (cfg.block_threads * (cfg.packed ? 2 : 1));
}

static void free_graph(GraphSlot& g)
{
    if (g.exec) cudaGraphExecDestroy(g.exec);
    if (g.graph) cudaGraphDestroy(g.graph);
    g = GraphSlot();
}

extern "C" int mppi_destroy(mppi_ctx* c)
{
    if (!c) return MPPI_OK;
    cudaDeviceSynchronize();
    free_graph(c->g_step); free_graph(c->g_opt);
    cudaFree(c->d_gates); cudaFree(c->d_ref); cudaFree(c->d_path); cudaFree(c->d_du);
    cudaFree(c->d_partials); cudaFree(c->d_headers); cudaFree(c->d_counters); cudaFree(c->d_hint);
    if (c->h_pin) cudaFreeHost(c->h_pin);
    cudaFree(c->d_in);
    cudaFree(c->d_hx0); cudaFree(c->d_hstart); cudaFree(c->d_hu); cudaFree(c->d_hcost); cudaFree(c->d_hw);
    delete c;
    return MPPI_OK;
}

template <typename T>
static cudaError_t dev_alloc(mppi_ctx* c, T** p, size_t n)
{
    cudaError_t e = cudaMalloc(reinterpret_cast<void**>(p), n * sizeof(T));
    if (e == cudaSuccess) c->scratch_bytes += (int64_t)(n * sizeof(T));
    return e;
}

extern "C" int mppi_create(const mppi_params* p, mppi_ctx** out)
{
    if (!p || !out) return fail(nullptr, MPPI_E_NULL, "mppi_create: NULL argument");
    *out = nullptr;
    int rc = validate(p);
    if (rc != MPPI_OK) return rc;
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0)
        return fail(nullptr, MPPI_E_CUDA, std::string("no CUDA device: ") + cudaGetErrorString(e));
    mppi_ctx* c = new (std::nothrow) mppi_ctx();
    if (!c) return fail(nullptr, MPPI_E_ALLOC, "host allocation failed");
    c->prm = *p;
    cudaGetDevice(&c->device);
    cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, c->device);
    cudaDeviceGetAttribute(&c->l2_bytes, cudaDevAttrL2CacheSize, c->device);

    // derived constants: computed in double from the fp32 parameters, rounded once
    DevParams& d = c->dp;
    std::memset(&d, 0, sizeof d);
    d.K = p->K; d.N = p->N; d.B = p->B; d.window = p->window;
    {
        const double h = (double)p->dt;
        d.h2 = (float)(h / 2); d.h3 = (float)(h / 3); d.h4 = (float)(h / 4); d.h6 = (float)(h / 6);
        d.h12 = (float)(h / 12); d.hh2 = (float)(h * h / 2); d.hh3 = (float)(h * h / 3);
    }
    d.dt = p->dt; d.inv_lambda = (float)(1.0 / (double)p->lambda); d.sigma = p->sigma;
    d.bm_k = (float)(-2.0 * 0.6931471805599453 * (double)p->sigma * (double)p->sigma);
    d.bm_kv = (float)(-2.0 * 0.6931471805599453 * (double)p->sigma_v * (double)p->sigma_v);
    d.T_min = p->T_min; d.T_max = p->T_max;
    d.inv_mass = (float)(1.0 / (double)p->mass); d.g = p->g;
    d.hover = (float)((double)p->mass * (double)p->g / 4.0);
    const double lever = (double)p->arm / std::sqrt(2.0);
    d.ltx = (float)(lever / p->Jx); d.lty = (float)(lever / p->Jy); d.ltz = (float)((double)p->c_tau / p->Jz);
    d.gyx = (float)(((double)p->Jy - p->Jz) / p->Jx);
    d.gyy = (float)(((double)p->Jz - p->Jx) / p->Jy);
    d.gyz = (float)(((double)p->Jx - p->Jy) / p->Jz);
    d.w_omega = p->w_omega; d.miss = p->gate_miss_penalty; d.bonus = p->gate_pass_bonus;
    d.q_near = p->q_near; d.r_near2 = (float)((double)p->r_near * (double)p->r_near); d.near_mode = p->near_mode;
    d.input_model = p->input_model; d.rate_max = p->rate_max;
    d.drag_x = p->drag_x; d.drag_y = p->drag_y; d.drag_z = p->drag_z;
    d.drag4_x = 4.0f * p->drag_x; d.drag4_y = 4.0f * p->drag_y; d.drag4_z = 4.0f * p->drag_z;
    d.drag_dd4 = (float)(4.0 * ((double)p->drag_z - (double)p->drag_x));
    d.inv_mass2 = 2.0f * d.inv_mass;                       // exact rescalings (fdyn_general, mppi_rate.cuh)
    d.w_limit = p->w_limit; d.omega_max = p->omega_max;
    d.sigma_v = p->sigma_v; d.dv_max = p->dv_max; d.v_theta_max = p->v_theta_max; d.r_dv = p->r_dv;
    d.Qp = p->Qp; d.Qv = p->Qv; d.Qq = p->Qq; d.Qw = p->Qw; d.R = p->R;
    d.q_c = p->q_contour; d.q_l = p->q_lag; d.mu = p->mu_progress;

    LaunchCfg& cfg = c->cfg;
    cfg.objective = p->objective; cfg.fast_math = p->fast_math ? 1 : 0;
    cfg.fused = p->pipeline == MPPI_PIPE_FUSED;
    cfg.store_du = (!cfg.fused || p->store_noise) ? 1 : 0;
    pick_shape(p, c->sm_count, &cfg.block_threads, &cfg.lat_consumers, &cfg.packed, &cfg.pipe, &cfg.scan);
    cfg.rate = p->input_model == 1;
    c->xdim = p->objective == MPPI_OBJ_CONTOUR_PAPER ? 19 : cfg.rate ? 17 : 13;
    d.blocks_per_ctrl = blocks_per_ctrl_of(p, cfg);
    // floats per partial, a multiple of 8: every 32-byte sector of a partial is then written completely
    d.part_stride = (4 * p->N + 4 + (p->objective == MPPI_OBJ_CONTOUR_PAPER ? p->N : 0) + 7) & ~7;
    cfg.pipe_shallow = 0;
    cfg.smem_bytes = 0;   // fixed once the track is known
    // input_model = 1: the pipelined latency kernel is the faster one for few rollouts, but its rings share the
    // shared memory with the track, which is not known yet: keep the scalar shape, size the partials for
    // either, and let prepare() switch once the track has been set
    c->scalar_tpb = cfg.block_threads; c->scalar_packed = cfg.packed;
    c->lazy_pipe = rate_pipe_candidate(p, c->sm_count) ? 1 : 0;
    d.pipe_d = 4; d.pipe_df = 3;
    // AUTO may move to another kernel once the track is known (prepare()): size the partials for the largest grid
    const int max_blocks = (c->lazy_pipe || p->variant == MPPI_VARIANT_AUTO) ? std::max(p->K / 32, d.blocks_per_ctrl) : d.blocks_per_ctrl;

    const size_t BN4 = (size_t)p->B * p->N * 4, BK = (size_t)p->B * p->K;
#define CKC(call)                                                        \
    do {                                                                 \
        cudaError_t e2_ = (call);                                        \
        if (e2_ != cudaSuccess) {                                        \
            int r_ = cuda_fail(nullptr, e2_, #call);                     \
            mppi_destroy(c);                                             \
            return r_;                                                   \
        }                                                                \
    } while (0)
    c->keep_du = cfg.store_du != 0;
    if (cfg.store_du) CKC(dev_alloc(c, &c->d_du, (size_t)p->B * p->N * p->K));
    if (cfg.fused) {
        CKC(dev_alloc(c, &c->d_partials, (size_t)p->B * max_blocks * d.part_stride));
        CKC(dev_alloc(c, &c->d_headers, (size_t)p->B * max_blocks));
        CKC(dev_alloc(c, &c->d_counters, (size_t)p->B + 1));
        CKC(cudaMemset(c->d_counters, 0, ((size_t)p->B + 1) * sizeof(unsigned)));
        CKC(dev_alloc(c, &c->d_hint, (size_t)p->B));
        CKC(cudaMemset(c->d_hint, 0, (size_t)p->B * sizeof(unsigned)));
    }
    CKC(dev_alloc(c, &c->d_hx0, (size_t)p->B * c->xdim));
    CKC(dev_alloc(c, &c->d_hstart, (size_t)p->B));
    CKC(dev_alloc(c, &c->d_hu, BN4));
    CKC(dev_alloc(c, &c->d_hcost, BK));
    CKC(dev_alloc(c, &c->d_hw, BK));
#undef CKC
    if (cfg.fused) {
        // layout of the mapped staging block, every part 256-byte aligned
        auto up = [](size_t v) { return (v + 255) & ~(size_t)255; };
        size_t o = 0;
        c->pin_x0 = o; o = up(o + (size_t)p->B * c->xdim * sizeof(float));
        c->pin_start = o; o = up(o + (size_t)p->B * sizeof(int32_t));
        c->pin_u = o; o = up(o + BN4 * sizeof(float));
        c->pin_unew = o; o = up(o + BN4 * sizeof(float));
        c->pin_cost = o; o = up(o + BK * sizeof(float));
        c->pin_w = o; o = up(o + BK * sizeof(float));
        c->pin_flag = o; o = up(o + sizeof(unsigned));
        c->pin_bytes = o;
        void* hp = nullptr; void* dp = nullptr;
        if (cudaHostAlloc(&hp, o, cudaHostAllocMapped) == cudaSuccess &&
            cudaHostGetDevicePointer(&dp, hp, 0) == cudaSuccess) {
            c->h_pin = (unsigned char*)hp; c->d_pin = (unsigned char*)dp;
            std::memset(hp, 0, o);
            if (dev_alloc(c, &c->d_in, c->pin_unew) != cudaSuccess) {
                cudaGetLastError(); cudaFreeHost(hp); c->h_pin = nullptr; c->d_in = nullptr;
            }
        } else {
            if (hp) cudaFreeHost(hp);
            cudaGetLastError();          // mapping unavailable: mppi_step_host uses explicit copies
        }
    }
    *out = c;
    return MPPI_OK;
}

// ---- tracks -------------------------------------------------------------------------------------

static int upload_f4(mppi_ctx* c, float4** dst, const std::vector<float4>& v)
{
    if (*dst) { cudaDeviceSynchronize(); cudaFree(*dst); *dst = nullptr; }
    CK(c, dev_alloc(c, dst, v.size()));
    CK(c, cudaMemcpy(*dst, v.data(), v.size() * sizeof(float4), cudaMemcpyHostToDevice));
    free_graph(c->g_step); free_graph(c->g_opt);   // shared-memory size may have changed
    return MPPI_OK;
}

extern "C" int mppi_set_gates(mppi_ctx* c, const float* g, int G)
{
    if (!c || !g) return fail(c, MPPI_E_NULL, "mppi_set_gates: NULL argument");
    if (G < 1 || G > MPPI_MAX_GATES) return fail(c, MPPI_E_TRACK, "G must be in 1..MPPI_MAX_GATES");
    std::vector<float4> v(4 * (size_t)G);
    for (int i = 0; i < G; ++i) {
        const float* r = g + 11 * i;
        for (int j = 0; j < 11; ++j)
            if (!std::isfinite(r[j])) return fail(c, MPPI_E_TRACK, "gate entry is not finite");
        const double n[3] = {r[3], r[4], r[5]}, h[3] = {r[6], r[7], r[8]};
        const double nn = std::sqrt(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]);
        const double hh = std::sqrt(h[0] * h[0] + h[1] * h[1] + h[2] * h[2]);
        const double nh = n[0] * h[0] + n[1] * h[1] + n[2] * h[2];
        if (std::fabs(nn - 1.0) > 1e-4 || std::fabs(hh - 1.0) > 1e-4 || std::fabs(nh) > 1e-4)
            return fail(c, MPPI_E_TRACK, "gate normal / in-plane axis must be unit and orthogonal (1e-4)");
        if (!(r[9] > 0.0f) || !(r[10] > 0.0f)) return fail(c, MPPI_E_TRACK, "gate half-sizes must be > 0");
        const double vx = h[1] * n[2] - h[2] * n[1], vy = h[2] * n[0] - h[0] * n[2], vz = h[0] * n[1] - h[1] * n[0];
        v[4 * i + 0] = make_float4(r[0], r[1], r[2], r[9]);
        v[4 * i + 1] = make_float4(r[3], r[4], r[5], r[10]);
        const double nc = n[0] * (double)r[0] + n[1] * (double)r[1] + n[2] * (double)r[2];   // plane offset n . c
        v[4 * i + 2] = make_float4(r[6], r[7], r[8], (float)nc);
        v[4 * i + 3] = make_float4((float)vx, (float)vy, (float)vz, 0.0f);
    }
    int rc = upload_f4(c, &c->d_gates, v);
    if (rc) return rc;
    c->dp.G = G; c->dp.gates = c->d_gates; c->have_gates = true;
    return MPPI_OK;
}

extern "C" int mppi_set_reference(mppi_ctx* c, const float* ref, int M)
{
    if (!c || !ref) return fail(c, MPPI_E_NULL, "mppi_set_reference: NULL argument");
    if (M < c->prm.N + 1) return fail(c, MPPI_E_TRACK, "reference needs at least N+1 rows");
    std::vector<float4> v(4 * (size_t)M);
    for (int i = 0; i < M; ++i) {
        const float* r = ref + 13 * i;
        for (int j = 0; j < 13; ++j)
            if (!std::isfinite(r[j])) return fail(c, MPPI_E_TRACK, "reference entry is not finite");
        v[4 * i + 0] = make_float4(r[0], r[1], r[2], r[3]);
        v[4 * i + 1] = make_float4(r[4], r[5], r[6], r[7]);
        v[4 * i + 2] = make_float4(r[8], r[9], r[10], r[11]);
        v[4 * i + 3] = make_float4(r[12], 0.0f, 0.0f, 0.0f);
    }
    int rc = upload_f4(c, &c->d_ref, v);
    if (rc) return rc;
    c->dp.M = M; c->dp.ref = c->d_ref; c->have_ref = true;
    return MPPI_OK;
}

extern "C" int mppi_set_path(mppi_ctx* c, const float* pts, int P, int closed)
{
    if (!c || !pts) return fail(c, MPPI_E_NULL, "mppi_set_path: NULL argument");
    if (P < 2 * c->prm.window + 1 || P > MPPI_MAX_PATH)
        return fail(c, MPPI_E_TRACK, "P must be in 2*window+1..MPPI_MAX_PATH");
    for (int i = 0; i < 3 * P; ++i)
        if (!std::isfinite(pts[i])) return fail(c, MPPI_E_TRACK, "path entry is not finite");
    // [R-22] arc length = cumulative chord length, tangent = normalised central difference;
    // computed in double from the fp32 points, rounded once
    std::vector<double> s(P, 0.0);
    auto dist = [&](int a, int b) {
        double d0 = (double)pts[3 * a] - pts[3 * b], d1 = (double)pts[3 * a + 1] - pts[3 * b + 1],
               d2 = (double)pts[3 * a + 2] - pts[3 * b + 2];
        return std::sqrt(d0 * d0 + d1 * d1 + d2 * d2);
    };
    for (int i = 1; i < P; ++i) {
        const double d = dist(i, i - 1);
        if (!(d > 0.0)) return fail(c, MPPI_E_TRACK, "consecutive path points coincide");
        s[i] = s[i - 1] + d;
    }
    double L = s[P - 1];
    if (closed) {
        const double d = dist(0, P - 1);
        if (!(d > 0.0)) return fail(c, MPPI_E_TRACK, "closed path repeats its first point");
        L += d;
    }
    std::vector<float4> v(2 * (size_t)P);
    for (int i = 0; i < P; ++i) {
        int ip = i + 1, im = i - 1;
        if (closed) { ip %= P; im = (im + P) % P; }
        else { ip = ip > P - 1 ? P - 1 : ip; im = im < 0 ? 0 : im; }
        double t[3];
        for (int a = 0; a < 3; ++a) t[a] = (double)pts[3 * ip + a] - pts[3 * im + a];
        const double nt = std::sqrt(t[0] * t[0] + t[1] * t[1] + t[2] * t[2]);
        if (!(nt > 0.0)) return fail(c, MPPI_E_TRACK, "degenerate path tangent");
        // all points first, then all tangents: the nearest-vertex search reads points only, at a 16-byte stride
        v[i] = make_float4(pts[3 * i], pts[3 * i + 1], pts[3 * i + 2], (float)s[i]);
        v[(size_t)P + i] = make_float4((float)(t[0] / nt), (float)(t[1] / nt), (float)(t[2] / nt), 0.0f);
    }
    int rc = upload_f4(c, &c->d_path, v);
    if (rc) return rc;
    c->dp.P = P; c->dp.closed = closed ? 1 : 0; c->dp.path = c->d_path;
    c->dp.path_L = (float)L; c->dp.inv_path_L = (float)(1.0 / L);
    c->have_path = true;
    return MPPI_OK;
}

// ---- launch preparation ---------------------------------------------------------------------------

static int prepare(mppi_ctx* c)
{
    const int obj = c->prm.objective;
    if (((obj == MPPI_OBJ_GATE || obj == MPPI_OBJ_GATE_PAPER) && !c->have_gates) || (obj == MPPI_OBJ_TRACK && !c->have_ref) ||
        ((obj == MPPI_OBJ_CONTOUR || obj == MPPI_OBJ_CONTOUR_PAPER) && !c->have_path))
        return fail(c, MPPI_E_NO_TRACK, "mppi_set_gates / mppi_set_reference / mppi_set_path not called for this objective");
    if (obj == MPPI_OBJ_CONTOUR_PAPER && (!c->d_v_nom || !c->d_v_new))
        return fail(c, MPPI_E_NO_TRACK, "mppi_set_progress not called (MPPI_OBJ_CONTOUR_PAPER)");
    if (c->lazy_pipe) {
        // deep rings (4, 3) with at most one block per SM, or shallow rings (2, 2) and two blocks per SM for
        // grids up to twice the SM count; an explicit PIPELINED request takes whichever fits
        const bool force = c->prm.variant == MPPI_VARIANT_PIPELINED;
        const int64_t grid = (int64_t)c->prm.B * c->prm.K / 32;
        LaunchCfg pc = c->cfg; pc.pipe = 1; pc.block_threads = 320;
        DevParams pd = c->dp; pd.blocks_per_ctrl = c->prm.K / 32;
        int use_d = 0, use_df = 0;
        pd.pipe_d = 4; pd.pipe_df = 3;
        const bool deep = rollout_smem_bytes(pd, pc) <= 227 * 1024;
        pd.pipe_d = 2; pd.pipe_df = 2;
        const bool shallow2 = 2 * (rollout_smem_bytes(pd, pc) + 1024) <= 228 * 1024;
        if (deep && (grid <= c->sm_count || (force && !shallow2))) { use_d = 4; use_df = 3; }
        else if (shallow2 && (grid <= 2 * (int64_t)c->sm_count || force)) { use_d = 2; use_df = 2; }
        else if (deep && force) { use_d = 4; use_df = 3; }
        if (force && !use_d) return fail(c, MPPI_E_PARAM, "PIPELINED: track + horizon do not fit in shared memory beside the rings");
        const bool on = use_d != 0;
        if (on != (c->cfg.pipe == 1) || (on && (c->dp.pipe_d != use_d || c->dp.pipe_df != use_df))) {
            c->cfg.pipe = on ? 1 : 0;
            c->cfg.block_threads = on ? 320 : c->scalar_tpb;
            c->cfg.packed = on ? 0 : c->scalar_packed;
            c->dp.blocks_per_ctrl = on ? c->prm.K / 32 : c->prm.K / (c->scalar_tpb * (c->scalar_packed ? 2 : 1));
            if (on) { c->dp.pipe_d = use_d; c->dp.pipe_df = use_df; c->cfg.pipe_shallow = use_d == 2; }
            c->cfg.smem_bytes = 0;
        }
    }
    // latency kernel under search-contouring: the rollout / search split needs a position table in shared memory
    c->cfg.lat_split = (c->cfg.lat_consumers > 0 && obj == MPPI_OBJ_CONTOUR) ? 1 : 0;
    size_t need = rollout_smem_bytes(c->dp, c->cfg);
    if (c->cfg.lat_split && need > 227 * 1024) { c->cfg.lat_split = 0; need = rollout_smem_bytes(c->dp, c->cfg); }
    if (need > 227 * 1024 && c->prm.variant == MPPI_VARIANT_AUTO && c->prm.input_model == 0 &&
        (c->cfg.pipe || c->cfg.lat_consumers || c->cfg.scan)) {
        // the kernel picked from the warp count alone does not fit with this track: next choice of pick_shape
        for (int avoid : {1, 3}) {
            if (avoid == 1 && !c->cfg.pipe && !c->cfg.scan) continue;
            LaunchCfg nc = c->cfg;
            pick_shape(&c->prm, c->sm_count, &nc.block_threads, &nc.lat_consumers, &nc.packed, &nc.pipe, &nc.scan, avoid);
            DevParams nd = c->dp;
            nd.blocks_per_ctrl = blocks_per_ctrl_of(&c->prm, nc);
            const size_t nn = rollout_smem_bytes(nd, nc);
            if (nn <= 227 * 1024 || avoid == 3) {
                c->cfg = nc; c->cfg.smem_bytes = 0; c->dp.blocks_per_ctrl = nd.blocks_per_ctrl; need = nn;
                if (!nc.lat_consumers) c->cfg.lat_split = 0;
                free_graph(c->g_step); free_graph(c->g_opt);
                break;
            }
        }
    }
    // fused throughput kernels: scratch for dU, used only in iterations that follow one with many weight-carrying
    // samples (StepArgs::hint).  If the allocation fails the kernels simply keep re-deriving the noise.
    if (c->cfg.fused && !c->cfg.pipe && !c->cfg.scan && !c->cfg.lat_consumers && c->prm.objective != MPPI_OBJ_CONTOUR_PAPER && !c->d_du &&
        !c->du_tried) {
        c->du_tried = true;
        // at most 1 GiB of such scratch (configs[4]: 210 MB); larger batches keep re-deriving the noise
        const size_t n_du = (size_t)c->prm.B * c->prm.N * c->prm.K;
        if (n_du * sizeof(float4) <= ((size_t)1 << 30) && dev_alloc(c, &c->d_du, n_du) != cudaSuccess) { cudaGetLastError(); c->d_du = nullptr; }
    }
    if (need != c->cfg.smem_bytes) {
        if (need > 227 * 1024) return fail(c, MPPI_E_PARAM, "track + horizon do not fit in shared memory");
        if (need > 48 * 1024)
            CK(c, cudaFuncSetAttribute(rollout_kernel_ptr(c->cfg), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)need));
        c->cfg.smem_bytes = need;
    }
    return MPPI_OK;
}

static bool overlaps(const void* a, size_t na, const void* b, size_t nb)
{
    const char* x = (const char*)a; const char* y = (const char*)b;
    return x < y + nb && y < x + na;
}

static StepArgs make_args(mppi_ctx* c, const float* x0, const int32_t* start, const float* u_nom,
                          uint64_t seed, uint32_t iter, float* u_new, float* cost, float* w)
{
    StepArgs a;
    a.x0 = x0; a.start = start; a.u_nom = u_nom; a.u_new = u_new; a.cost = cost; a.weights = w;
    a.du = c->d_du; a.partials = c->d_partials; a.headers = c->d_headers; a.counters = c->d_counters;
    a.hint = (c->cfg.fused && !c->cfg.pipe && !c->cfg.scan && !c->cfg.lat_consumers && c->d_du) ? c->d_hint : nullptr;
    a.prev_front = c->d_prev_front; a.v_nom = c->d_v_nom; a.v_new = c->d_v_new;
    a.done_flag = nullptr; a.done_value = 0; a.pdl = 0;
#ifdef MPPI_TIMELINE
    {
        static unsigned long long* tl = nullptr;      // profiling builds only: one buffer, read back by the probe script
        if (!tl) { cudaMalloc(&tl, 16 * 65536 * sizeof(unsigned long long)); cudaMemset(tl, 0, 16 * 65536 * sizeof(unsigned long long)); }
        a.timeline = tl;
    }
#endif
    a.seed_lo = (uint32_t)(seed & 0xffffffffu); a.seed_hi = (uint32_t)(seed >> 32); a.iter = iter;
    for (uint32_t r = 0; r < 10; ++r) {          // Philox key schedule (Weyl sequence), hoisted out of the kernel
        a.rk[2 * r] = a.seed_lo + r * 0x9E3779B9u;
        a.rk[2 * r + 1] = a.seed_hi + r * 0xBB67AE85u;
    }
    return a;
}

static int enqueue_iteration(mppi_ctx* c, const StepArgs& a, cudaStream_t s, bool pdl = false)
{
    CK(c, launch_rollout(c->dp, a, c->cfg, s, pdl));
    c->launches += 1;
    if (!c->cfg.fused) {
        CK(c, launch_reduce(c->dp, a, s));
        c->launches += 1;
    }
    return MPPI_OK;
}

static void node_params(mppi_ctx* c, bool reduce, void** kp, cudaKernelNodeParams* np)
{
    std::memset(np, 0, sizeof *np);
    if (!reduce) {
        np->func = const_cast<void*>(rollout_kernel_ptr(c->cfg));
        np->gridDim = dim3(c->dp.blocks_per_ctrl, c->dp.B);
        np->blockDim = dim3(c->cfg.block_threads);
        np->sharedMemBytes = (unsigned)c->cfg.smem_bytes;
    } else {
        np->func = const_cast<void*>(reduce_kernel_ptr());
        np->gridDim = dim3(c->dp.N, c->dp.B);
        np->blockDim = dim3(kReduceThreads);
        np->sharedMemBytes = 0;
    }
    np->kernelParams = kp;
}

// Build (once) a graph of n iterations; every replay only rewrites the kernel parameters.
static int graph_run(mppi_ctx* c, GraphSlot& g, const std::vector<StepArgs>& args, cudaStream_t s)
{
    const int n = (int)args.size();
    DevParams dp = c->dp;
    const bool build = !g.exec || g.n_iters != n;
    if (build) {
        free_graph(g);
        CK(c, cudaGraphCreate(&g.graph, 0));
    }
    cudaGraphNode_t prev = nullptr;
    for (int i = 0; i < n; ++i) {
        StepArgs a = args[i];
        int lat_c = c->cfg.lat_consumers | (c->cfg.lat_split << 8);
        void* kp[3] = {&dp, &a, &lat_c};
        cudaKernelNodeParams np;
        for (int pass = 0; pass < (c->cfg.fused ? 1 : 2); ++pass) {
            node_params(c, pass == 1, kp, &np);
            std::vector<cudaGraphNode_t>& nodes = pass ? g.reduce_nodes : g.rollout_nodes;
            if (build) {
                cudaGraphNode_t node;
                CK(c, cudaGraphAddKernelNode(&node, g.graph, prev ? &prev : nullptr, prev ? 1 : 0, &np));
                nodes.push_back(node);
                prev = node;
            } else {
                CK(c, cudaGraphExecKernelNodeSetParams(g.exec, nodes[i], &np));
            }
        }
    }
    if (build) {
        CK(c, cudaGraphInstantiate(&g.exec, g.graph, 0));
        g.n_iters = n;
    }
    CK(c, cudaGraphLaunch(g.exec, s));
    c->launches += (int64_t)n * (c->cfg.fused ? 1 : 2);
    return MPPI_OK;
}

extern "C" int mppi_step(mppi_ctx* c, const float* d_x0, const int32_t* d_start, const float* d_u_nom,
                         uint64_t seed, uint32_t iter, float* d_u_new, float* d_cost, float* d_weights,
                         void* stream)
{
    if (!c) return MPPI_E_NULL;
    if (!d_x0 || !d_start || !d_u_nom || !d_u_new || !d_cost || !d_weights)
        return fail(c, MPPI_E_NULL, "mppi_step: NULL device pointer");
    const size_t ub = (size_t)c->prm.B * c->prm.N * 4 * sizeof(float);
    if (d_u_new != d_u_nom && overlaps(d_u_new, ub, d_u_nom, ub))
        return fail(c, MPPI_E_RANGE, "d_u_new partially overlaps d_u_nom");
    int rc = prepare(c);
    if (rc) return rc;
    const StepArgs a = make_args(c, d_x0, d_start, d_u_nom, seed, iter, d_u_new, d_cost, d_weights);
    if (c->prm.use_graph) return graph_run(c, c->g_step, std::vector<StepArgs>(1, a), (cudaStream_t)stream);
    return enqueue_iteration(c, a, (cudaStream_t)stream);
}

extern "C" int mppi_optimize(mppi_ctx* c, const float* d_x0, const int32_t* d_start, float* d_u,
                             uint64_t seed, uint32_t iter0, int n_iters, float* d_cost, float* d_weights,
                             void* stream)
{
    if (!c) return MPPI_E_NULL;
    if (!d_x0 || !d_start || !d_u || !d_cost || !d_weights)
        return fail(c, MPPI_E_NULL, "mppi_optimize: NULL device pointer");
    if (n_iters < 1 || n_iters > 1024) return fail(c, MPPI_E_RANGE, "n_iters must be in 1..1024");
    if (c->prm.objective == MPPI_OBJ_CONTOUR_PAPER && c->d_v_nom != c->d_v_new)
        return fail(c, MPPI_E_RANGE, "mppi_optimize under MPPI_OBJ_CONTOUR_PAPER needs mppi_set_progress(v, v) (in place)");
    int rc = prepare(c);
    if (rc) return rc;
    std::vector<StepArgs> args;
    for (int i = 0; i < n_iters; ++i)
        args.push_back(make_args(c, d_x0, d_start, d_u, seed, iter0 + (uint32_t)i, d_u, d_cost, d_weights));
    if (c->prm.use_graph) return graph_run(c, c->g_opt, args, (cudaStream_t)stream);
    // plain launches.  The pipelined kernel chains its iterations by programmatic dependent launch: every iteration
    // lets the next one start on the SMs once its rollouts are done, and the next one stages its track and draws the
    // state-independent half of its noise while this one publishes and combines, then waits (griddepcontrol.wait)
    // before it reads the nominal.  Bit-identical results (tests: optimize == chain of steps).
    const bool pdl = (c->cfg.pipe || c->cfg.scan) && !c->cfg.rate && c->cfg.fused && n_iters > 1;
    for (int i = 0; i < n_iters; ++i) {
        if (pdl) args[i].pdl = (i > 0 ? 1 : 0) | (i + 1 < n_iters ? 2 : 0);
        rc = enqueue_iteration(c, args[i], (cudaStream_t)stream, pdl && i > 0);
        if (rc) return rc;
    }
    return MPPI_OK;
}

extern "C" int mppi_step_host(mppi_ctx* c, const float* h_x0, const int32_t* h_start, const float* h_u_nom,
                              uint64_t seed, uint32_t iter, float* h_u_new, float* h_cost, float* h_weights,
                              void* stream)
{
    if (!c) return MPPI_E_NULL;
    if (!h_x0 || !h_start || !h_u_nom || !h_u_new) return fail(c, MPPI_E_NULL, "mppi_step_host: NULL host pointer");
    if (c->prm.objective == MPPI_OBJ_CONTOUR_PAPER)
        return fail(c, MPPI_E_PARAM, "mppi_step_host: not available for MPPI_OBJ_CONTOUR_PAPER (its progress column lives on the device)");
    cudaStream_t s = (cudaStream_t)stream;
    const size_t B = c->prm.B, N = c->prm.N, K = c->prm.K;
    if (c->h_pin) {
        // inputs: packed in pinned memory, one copy down.  outputs: u_new (and cost / weights when asked
        // for) are written into mapped host memory by the kernel itself, whose last block raises a
        // sequence number this thread polls -- no copy back, no stream synchronisation
        int rc = prepare(c);
        if (rc) return rc;
        unsigned char* hp = c->h_pin; unsigned char* dp = c->d_pin;
        std::memcpy(hp + c->pin_x0, h_x0, B * c->xdim * sizeof(float));
        std::memcpy(hp + c->pin_start, h_start, B * sizeof(int32_t));
        std::memcpy(hp + c->pin_u, h_u_nom, B * N * 4 * sizeof(float));
        CK(c, cudaMemcpyAsync(c->d_in, hp, c->pin_u + B * N * 4 * sizeof(float), cudaMemcpyHostToDevice, s));
        const unsigned char* di = c->d_in;
        StepArgs a = make_args(c, (const float*)(di + c->pin_x0), (const int32_t*)(di + c->pin_start),
                               (const float*)(di + c->pin_u), seed, iter, (float*)(dp + c->pin_unew),
                               h_cost ? (float*)(dp + c->pin_cost) : c->d_hcost,
                               h_weights ? (float*)(dp + c->pin_w) : c->d_hw);
        volatile unsigned* flag = (volatile unsigned*)(hp + c->pin_flag);
        const unsigned seq = ++c->host_seq ? c->host_seq : ++c->host_seq;     // never 0
        a.done_flag = (unsigned*)(dp + c->pin_flag); a.done_value = seq;
        rc = enqueue_iteration(c, a, s);
        if (rc) return rc;
        const auto t0 = std::chrono::steady_clock::now();
        unsigned spins = 0;
        while (*flag != seq) {
            if ((++spins & 0x3fff) == 0) {
                // every so often: has the stream failed, or is this taking implausibly long?
                const cudaError_t q = cudaStreamQuery(s);
                if (q != cudaSuccess && q != cudaErrorNotReady) return cuda_fail(c, q, "mppi_step_host: kernel");
                if (std::chrono::steady_clock::now() - t0 > std::chrono::seconds(10)) {
                    CK(c, cudaStreamSynchronize(s));
                    if (*flag != seq) return fail(c, MPPI_E_CUDA, "mppi_step_host: completion flag never arrived");
                }
            }
        }
        std::atomic_thread_fence(std::memory_order_acquire);
        std::memcpy(h_u_new, hp + c->pin_unew, B * N * 4 * sizeof(float));
        if (h_cost) std::memcpy(h_cost, hp + c->pin_cost, B * K * sizeof(float));
        if (h_weights) std::memcpy(h_weights, hp + c->pin_w, B * K * sizeof(float));
        return MPPI_OK;
    }
    CK(c, cudaMemcpyAsync(c->d_hx0, h_x0, B * c->xdim * sizeof(float), cudaMemcpyHostToDevice, s));
    CK(c, cudaMemcpyAsync(c->d_hstart, h_start, B * sizeof(int32_t), cudaMemcpyHostToDevice, s));
    CK(c, cudaMemcpyAsync(c->d_hu, h_u_nom, B * N * 4 * sizeof(float), cudaMemcpyHostToDevice, s));
    int rc = mppi_step(c, c->d_hx0, c->d_hstart, c->d_hu, seed, iter, c->d_hu, c->d_hcost, c->d_hw, stream);
    if (rc) return rc;
    CK(c, cudaMemcpyAsync(h_u_new, c->d_hu, B * N * 4 * sizeof(float), cudaMemcpyDeviceToHost, s));
    if (h_cost) CK(c, cudaMemcpyAsync(h_cost, c->d_hcost, B * K * sizeof(float), cudaMemcpyDeviceToHost, s));
    if (h_weights) CK(c, cudaMemcpyAsync(h_weights, c->d_hw, B * K * sizeof(float), cudaMemcpyDeviceToHost, s));
    CK(c, cudaStreamSynchronize(s));
    return MPPI_OK;
}

extern "C" int mppi_sim_step(mppi_ctx* c, float* d_x, int32_t* d_start, const float* d_u_new,
                             float* d_u_nom_next, void* stream)
{
    if (!c) return MPPI_E_NULL;
    if (!d_x || !d_start || !d_u_new || !d_u_nom_next) return fail(c, MPPI_E_NULL, "mppi_sim_step: NULL device pointer");
    if (c->prm.objective == MPPI_OBJ_CONTOUR_PAPER)
        return fail(c, MPPI_E_PARAM, "mppi_sim_step: MPPI_OBJ_CONTOUR_PAPER has rows of 19 and a fifth column: use mppi_sim_step_progress");
    const size_t ub = (size_t)c->prm.B * c->prm.N * 4 * sizeof(float);
    if (d_u_nom_next != d_u_new && overlaps(d_u_nom_next, ub, d_u_new, ub))
        return fail(c, MPPI_E_RANGE, "d_u_nom_next partially overlaps d_u_new");
    int rc = prepare(c);
    if (rc) return rc;
    CK(c, launch_sim(c->dp, c->prm.objective, d_x, d_start, d_u_new, d_u_nom_next, (cudaStream_t)stream));
    c->launches += 1;
    return MPPI_OK;
}

extern "C" int mppi_sim_step_progress(mppi_ctx* c, float* d_x, const float* d_u_new, float* d_u_nom_next,
                                      const float* d_v_new, float* d_v_nom_next, void* stream)
{
    if (!c) return MPPI_E_NULL;
    if (c->prm.objective != MPPI_OBJ_CONTOUR_PAPER)
        return fail(c, MPPI_E_PARAM, "mppi_sim_step_progress: the objective is not MPPI_OBJ_CONTOUR_PAPER");
    if (!d_x || !d_u_new || !d_u_nom_next || !d_v_new || !d_v_nom_next)
        return fail(c, MPPI_E_NULL, "mppi_sim_step_progress: NULL device pointer");
    const size_t ub = (size_t)c->prm.B * c->prm.N * 4 * sizeof(float), vb = ub / 4;
    if ((d_u_nom_next != d_u_new && overlaps(d_u_nom_next, ub, d_u_new, ub)) ||
        (d_v_nom_next != d_v_new && overlaps(d_v_nom_next, vb, d_v_new, vb)))
        return fail(c, MPPI_E_RANGE, "an output partially overlaps its input");
    CK(c, launch_sim_progress(c->dp, d_x, d_u_new, d_u_nom_next, d_v_new, d_v_nom_next, (cudaStream_t)stream));
    c->launches += 1;
    return MPPI_OK;
}

extern "C" int mppi_set_progress(mppi_ctx* c, const float* d_v_nom, float* d_v_new)
{
    if (!c) return MPPI_E_NULL;
    if (c->prm.objective != MPPI_OBJ_CONTOUR_PAPER)
        return fail(c, MPPI_E_PARAM, "mppi_set_progress: the objective is not MPPI_OBJ_CONTOUR_PAPER");
    if (!d_v_nom || !d_v_new) return fail(c, MPPI_E_NULL, "mppi_set_progress: NULL device pointer");
    c->d_v_nom = d_v_nom; c->d_v_new = d_v_new;
    return MPPI_OK;
}

extern "C" int mppi_set_prev_front(mppi_ctx* c, const int32_t* d_prev_front)
{
    if (!c) return MPPI_E_NULL;
    if (c->prm.objective != MPPI_OBJ_GATE_PAPER)
        return fail(c, MPPI_E_PARAM, "mppi_set_prev_front: the objective is not MPPI_OBJ_GATE_PAPER");
    c->d_prev_front = d_prev_front;
    return MPPI_OK;
}

extern "C" int mppi_front_flags(mppi_ctx* c, const float* d_x0, const int32_t* d_start, const float* d_u,
                                int32_t* d_front_out, void* stream)
{
    if (!c) return MPPI_E_NULL;
    if (!d_x0 || !d_start || !d_u || !d_front_out) return fail(c, MPPI_E_NULL, "mppi_front_flags: NULL device pointer");
    if (!c->have_gates) return fail(c, MPPI_E_NO_TRACK, "mppi_front_flags: mppi_set_gates not called");
    CK(c, launch_front(c->dp, d_x0, d_start, d_u, d_front_out, (cudaStream_t)stream));
    c->launches += 1;
    return MPPI_OK;
}

extern "C" const float* mppi_debug_noise(mppi_ctx* c) { return (c && c->keep_du) ? reinterpret_cast<const float*>(c->d_du) : nullptr; }

extern "C" int64_t mppi_launch_count(mppi_ctx* c) { return c ? c->launches : 0; }

#ifdef MPPI_TIMELINE
extern "C" MPPI_API int mppi_timeline_read(mppi_ctx* c, unsigned long long* host_out, int blocks)
{
    StepArgs a = make_args(c, nullptr, nullptr, nullptr, 0, 0, nullptr, nullptr, nullptr);
    cudaDeviceSynchronize();
    return cudaMemcpy(host_out, a.timeline, (size_t)blocks * 16 * sizeof(unsigned long long), cudaMemcpyDeviceToHost) == cudaSuccess ? 0 : -6;
}
#endif

extern "C" int mppi_get_info(mppi_ctx* c, mppi_info* o)
{
    if (!c || !o) return fail(c, MPPI_E_NULL, "mppi_get_info: NULL argument");
    if (o->struct_size != sizeof(mppi_info)) return fail(c, MPPI_E_PARAM, "mppi_info.struct_size mismatch");
    int rc = prepare(c);
    if (rc) return rc;
    cudaFuncAttributes fa;
    CK(c, cudaFuncGetAttributes(&fa, rollout_kernel_ptr(c->cfg)));
    int nb = 0;
    CK(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, rollout_kernel_ptr(c->cfg), c->cfg.block_threads,
                                                        c->cfg.smem_bytes));
    o->block_threads = c->cfg.block_threads;
    o->blocks_per_controller = c->dp.blocks_per_ctrl;
    o->grid_blocks = c->dp.blocks_per_ctrl * c->dp.B;
    o->regs_per_thread = fa.numRegs;
    o->static_smem_bytes = (int32_t)fa.sharedSizeBytes;
    o->dynamic_smem_bytes = (int32_t)c->cfg.smem_bytes;
    o->local_bytes_per_thread = (int32_t)fa.localSizeBytes;
    o->max_blocks_per_sm = nb;
    o->sm_count = c->sm_count;
    o->kernels_per_step = c->cfg.fused ? 1 : 2;
    o->samples_per_thread = c->cfg.packed ? 2 : 1;
    o->rollout_warps_per_block = c->cfg.scan ? 16 : c->cfg.pipe ? (c->cfg.rate ? 5 : 3) : c->cfg.lat_consumers ? c->cfg.lat_consumers : c->cfg.block_threads / 32;
    o->l2_bytes = c->l2_bytes;
    o->scratch_bytes = c->scratch_bytes;
    return MPPI_OK;
}
