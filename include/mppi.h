/*
 * mppi.h -- C ABI of libmppi: one MPPI iteration of the reference-free racing controller of
 * arXiv 2509.14726 as hand-written sm_100a CUDA kernels.
 *
 * What one call computes (BASELINE.json:north_star; Alg. 1), for each of B
 * independent controllers:
 *   1. K perturbed rotor-thrust sequences U^k = clamp(U* + dU^k), dU ~ N(0, sigma^2 I), drawn in
 *      the kernel from Philox4x32-10 with counter (sample k, step t, iter, controller b) and key
 *      = seed                                                     (eq.(3))
 *   2. each rolled out through RK4 quadrotor rigid-body dynamics over N steps of dt
 *                                                                  (eq.(2))
 *   3. each scored under one objective: gate progress with gate-plane crossing and target
 *      switching (eq.(6)), full-state tracking (eq.(8)) or
 *      contouring against an arc-length path (eq.(9)); or the paper's own gate
 *      objective with squared progress, Q_near term and temporal switching check (eq.(6),(7),
 *      Fig. 2)
 *   4. weights w_k = softmax(-J_k / lambda) and U*_new = sum_k w_k U^k
 *                                                     (eq.(4),(5))
 * The exact readings of every point the paper leaves open are listed in DESIGN.md (R-1..R-26).
 *
 * Conventions
 *   - Notation follows BASELINE.json: K samples, N horizon steps, B controllers (the paper
 *     writes M samples, K steps).
 *   - State x[13] = p(3), q(w,x,y,z) body->world, v(3) world, omega(3) body.  World z is up,
 *     gravity (0,0,-g).  Inputs are the four rotor thrusts in newtons.
 *   - All floating-point data is fp32, row-major, densely packed.  "device" pointers are CUDA
 *     device memory owned by the caller (e.g. torch tensors); "host" pointers are ordinary host
 *     memory, copied during the call.  The library never frees a caller pointer, and keeps one only
 *     until the work the call enqueued has run -- with three documented exceptions that stay
 *     registered until replaced: the flags of mppi_set_prev_front and the two columns of
 *     mppi_set_progress (the caller keeps them alive as long as mppi_step may run).
 *   - Every entry point returns MPPI_OK (0) or a negative mppi_status.  Nothing throws, aborts
 *     or prints.  NaN/Inf in device inputs are not detected; they propagate to the outputs.
 *     A SAMPLE whose rollout diverges (cost NaN or beyond the fp32 range) is reported with cost
 *     3.0e38 and gets weight 0; it does not spoil the other samples or u_new.
 *   - A context is not thread-safe; distinct contexts are independent.  All device work is
 *     enqueued on the cudaStream_t passed in (NULL = the legacy default stream) and is
 *     asynchronous with respect to the host unless stated otherwise.
 *   - A context owns ONE set of scratch buffers (block partials, tickets, staging, the optional dU
 *     array).  All calls on one context must therefore be stream-ordered: use one stream, or make
 *     every call wait (event dependency) for the previous call on that context.  Two calls of one
 *     context in flight on different streams race on that scratch and give wrong results.
 *   - There is no CPU fallback: without a CUDA device mppi_create fails with MPPI_E_CUDA.
 */
#ifndef MPPI_H_
#define MPPI_H_

#include <stdint.h>

#if defined(__GNUC__)
#define MPPI_API __attribute__((visibility("default")))
#else
#define MPPI_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mppi_ctx mppi_ctx; /* opaque, owned by the library */

typedef enum {
    MPPI_OBJ_GATE = 0,    /* J_gate,    eq.(6) PAPER.md:105-112 (BASELINE.json configs[0,1,4]) */
    MPPI_OBJ_TRACK = 1,   /* J_track,   eq.(8) PAPER.md:139-147 (configs[2])                   */
    MPPI_OBJ_CONTOUR = 2, /* J_contour, eq.(9) PAPER.md:149-161 (configs[3])                   */
    MPPI_OBJ_GATE_PAPER = 3, /* the paper's own J_gate: eq.(6),(7) PAPER.md:105-129 with squared distances,
                             the Q_near term and the temporal gate-switching check of Fig. 2
                             (PAPER.md:114-122); tracks are gates; see mppi_set_prev_front          */
    MPPI_OBJ_CONTOUR_PAPER = 4 /* the paper's own J_contour, eq.(9): the progress theta and
                             its speed v_theta are STATES (every x / x0 row has 19 entries: ..., T(4),
                             theta, v_theta), the progress acceleration is a FIFTH sampled input next to
                             the four thrust rates (so input_model must be 1), the path is looked up by
                             theta; fused pipeline only; see mppi_set_progress                      */
} mppi_objective;

typedef enum {
    MPPI_OK = 0,
    MPPI_E_NULL = -1,     /* a required pointer is NULL                                        */
    MPPI_E_PARAM = -2,    /* a parameter is out of range (see mppi_params)                     */
    MPPI_E_NO_TRACK = -3, /* mppi_step before the mppi_set_* call the objective needs          */
    MPPI_E_TRACK = -4,    /* track data rejected (see mppi_set_*)                              */
    MPPI_E_RANGE = -5,    /* buffers overlap partially, or a count is out of range             */
    MPPI_E_CUDA = -6,     /* a CUDA call failed; text from mppi_last_error                     */
    MPPI_E_ALLOC = -7     /* host or device allocation failed                                  */
} mppi_status;

typedef enum {
    MPPI_PIPE_FUSED = 0,   /* one kernel per iteration: rollout + cost + block-local softmax
                              partials + last-block combine; the perturbations never leave the SM
                              (they are re-derived from the counter-based stream where needed)  */
    MPPI_PIPE_TWO_PASS = 1 /* rollout kernel stores dU [B][N][K][4] to HBM, a second fused
                              min / exp-weight / weighted-sum kernel reads it back              */
} mppi_pipeline;

typedef enum {
    MPPI_VARIANT_AUTO = 0,       /* time-parallel kernel where it applies and B*K/32 <= the SM count, pipelined or
                                    latency kernel while B*K/32 warps cannot fill the chip, else packed (K % 64
                                    == 0) or scalar throughput (thresholds from the batch sweep, profiles/)    */
    MPPI_VARIANT_THROUGHPUT = 1, /* one sample per thread, noise drawn inside the horizon loop; block_threads
                                    samples per block                                                      */
    MPPI_VARIANT_LATENCY = 2,    /* 256-thread blocks: all warps draw the noise of 32 C samples into shared
                                    memory first, then C warps (C = 1, 2 or 4) roll out; fused pipeline only */
    MPPI_VARIANT_PIPELINED = 4,  /* latency kernel, 256-thread blocks of 32 samples: five warps draw the noise,
                                    three warps on three SM sub-partitions carry the body-rate, attitude and
                                    translation chains of the same rollouts, pipelined over the horizon steps
                                    through shared-memory rings (mbarriers); fused pipeline only.  Under
                                    input_model = 1: 320-thread blocks, five chains (thrust states + body
                                    rates, attitude, two warps for the drag matrices of the RK4 stages,
                                    velocity / position); N <= 100, every objective but the search-based
                                    contouring; under MPPI_OBJ_CONTOUR_PAPER the path must fit in shared memory
                                    beside the rings (else mppi_step -> MPPI_E_PARAM; AUTO then stays on the
                                    throughput kernel)                                                      */
    MPPI_VARIANT_PACKED = 3,     /* throughput kernel with TWO samples per thread held in packed fp32x2
                                    registers (sm_100a FFMA2); needs K % 64 == 0; costs are bit-identical
                                    to MPPI_VARIANT_THROUGHPUT.  Under input_model = 1: every objective but the
                                    search-based contouring, block_threads <= 128 (else MPPI_E_PARAM); AUTO
                                    takes it when B K / 32 >= 8 x the SM count                             */
    MPPI_VARIANT_SCAN = 5        /* time-parallel latency kernel (eq.(2) PAPER.md:65-72 as a cascade of linear
                                    recurrences): blocks of up to 32 samples x 16 lanes, every rollout split over
                                    16 lanes ALONG THE HORIZON; body rates, attitude, velocity and position of
                                    the chunks are joined by warp-shuffle scans (affine maps, quaternion
                                    products, sums).  Needs input_model = 0, Jx == Jy (then the body-rate
                                    equations are linear given the yaw rate), objective MPPI_OBJ_GATE or
                                    MPPI_OBJ_GATE_PAPER, N <= 64, the fused pipeline and block_threads 0 (else
                                    MPPI_E_PARAM).  Same RK4, same per-step
                                    renormalisation, another association order: states equal the other kernels'
                                    to rounding, not bit for bit.  Samples per block (28 for K = 4096 on 148
                                    SMs) follow the SM count, so the summation order of the update -- not the
                                    costs -- depends on the GPU model; on one GPU every call is deterministic.
                                    AUTO takes it for such configurations when B K / 32 <= the SM count       */
} mppi_variant;

/* Parameters of Alg. 1 (samples, horizon, lambda, Sigma) plus the model and cost
 * constants of BASELINE.json configs[0..3].  struct_size = sizeof(mppi_params) versions the ABI. */
typedef struct {
    uint32_t struct_size;
    int32_t K;         /* samples per controller; > 0 and a multiple of 32                       */
    int32_t N;         /* horizon steps; 1..MPPI_MAX_N                                           */
    int32_t B;         /* independent controllers; >= 1                                          */
    int32_t objective; /* mppi_objective                                                         */
    float dt;          /* s, > 0                                                                 */
    float lambda;      /* temperature of eq.(4), cost units, > 0                                 */
    float sigma;       /* per-rotor noise std, N, >= 0 (Sigma = sigma^2 I, eq.(3))               */
    float mass, Jx, Jy, Jz; /* kg, kg m^2 (diagonal inertia), all > 0                            */
    float arm;         /* m; lever of PAPER.md:70 is arm / sqrt(2)                               */
    float c_tau;       /* m; rotor torque coefficient of PAPER.md:70                             */
    float g;           /* m/s^2                                                                  */
    float T_min, T_max;/* per-rotor hard clamp, N, T_min <= T_max                                */
    float w_omega;     /* body-rate weight of the gate and contouring objectives                 */
    float gate_miss_penalty; /* added on a plane crossing outside the opening                    */
    float gate_pass_bonus;   /* subtracted on a valid pass                                       */
    float Qp, Qv, Qq, Qw, R; /* tracking weights of eq.(8); R acts on (T - m g / 4)              */
    float q_contour, q_lag, mu_progress; /* contouring weights of eq.(9)                         */
    int32_t window;    /* contouring nearest-vertex search half-width in points, 1..64           */
    int32_t pipeline;  /* mppi_pipeline                                                          */
    int32_t use_graph; /* 1: replay each step as a CUDA graph; 0: plain stream launches          */
    int32_t block_threads; /* threads per block of the rollout kernel: 0 = auto, else 32..256,
                              a multiple of 32 that divides K (packed variant: <= 128 and
                              2*block_threads divides K)                                                   */
    int32_t fast_math; /* 0: IEEE-accurate logf/sincospif/sqrtf/expf; 1: MUFU approximations for
                          the Box-Muller transform (error budget)                 */
    int32_t store_noise; /* 1: also keep dU of the last step for mppi_debug_noise (always kept
                            in the TWO_PASS pipeline)                                            */
    int32_t variant;   /* mppi_variant: which rollout kernel the fused pipeline launches          */
    float q_near, r_near; /* MPPI_OBJ_GATE_PAPER, eq.(7): + q_near |p_k - c|^2 on every pre-step state
                          within r_near metres of its target gate centre; both >= 0 (the paper
                          prints neither value)                                                  */
    int32_t input_model; /* 0: the inputs are the four rotor thrusts, x has 13 entries (configs).
                          1: the paper's own model: the inputs are the thrust RATES
                          dT/dt in N/s and the rotor thrusts are states: every x / x0 row has 17
                          entries (p, q, v, omega, T(4)); u_nom / u_new hold rates; sigma is in N/s.
                          Rates are clamped to [-rate_max, rate_max], the thrust states are
                          projected onto [T_min, T_max] after every step, eq.(8)'s input term
                          R |u|^2 acts on the rates.  Kernels: scalar throughput (THROUGHPUT) and
                          pipelined latency (PIPELINED); AUTO picks the latter when B*K/32 warps
                          fit one per SM; mppi_sim_step advances the 17-entry rows                */
    float rate_max;      /* N/s, > 0 when input_model = 1 (Table I: 10)            */
    float drag_x, drag_y, drag_z; /* D = diag(.) of eq.(2)'s rotor drag - R D R^T v, body frame, 1/s,
                          >= 0; input_model = 1 only (the paper prints no value)                  */
    float sigma_v;       /* MPPI_OBJ_CONTOUR_PAPER: std of the sampled progress acceleration, m/s^2, >= 0    */
    float dv_max;        /* its range [-dv_max, dv_max], > 0 (Table I: 20)                  */
    float v_theta_max;   /* 0 <= v_theta <= v_theta_max, > 0 (eq.(9); Table I: 10)                       */
    float r_dv;          /* weight of |Delta v_theta|^2 in eq.(9), >= 0                                  */
    float w_limit, omega_max; /* input_model = 1: soft body-rate limit ("external cost"):
                          + w_limit sum_i max(0, |omega_i| - omega_max)^2 on every post-step state */
    int32_t near_mode;   /* MPPI_OBJ_GATE_PAPER, eq.(7): the gate whose centre the near term measures
                          against.  0: the target gate of the step (a state that already targets the next gate is far
                          from it, so the term ends with the switch).  1: the horizon's START gate p0_gate, before and
                          after the switch ("prevent states near the current gate p0_gate ... from deviating too much
                          from it", read literally).  DESIGN.md readings R-24 / R-40                       */
} mppi_params;

#define MPPI_MAX_N 256
#define MPPI_MAX_GATES 64
#define MPPI_MAX_PATH 2048
#define MPPI_MAX_WINDOW 64

/* Fills *p with struct_size and the constants of BASELINE.json configs[0] (K=256, N=20, B=1). */
MPPI_API int mppi_default_params(mppi_params* p);

/* Validates *p (MPPI_E_PARAM names the first offender through mppi_last_error(NULL)), creates the
 * context on the current CUDA device and allocates its device scratch.  No kernel is launched. */
MPPI_API int mppi_create(const mppi_params* p, mppi_ctx** out);
MPPI_API int mppi_destroy(mppi_ctx* ctx); /* synchronises the device, frees everything; NULL is accepted */

/* Waypoints W of Alg. 1.  host_gates [G][11]: centre c(3), unit normal n(3) = the
 * direction of travel, unit in-plane axis h(3) with n.h = 0, half-width along h, half-height
 * along v = h x n.  1 <= G <= MPPI_MAX_GATES.  MPPI_E_TRACK if |n|,|h| differ from 1 or n.h from
 * 0 by more than 1e-4, or a half-size is <= 0.  Synchronous host->device copy. */
MPPI_API int mppi_set_gates(mppi_ctx* ctx, const float* host_gates, int G);

/* Reference trajectory tau_ref of Alg. 1.  host_ref [M][13], one full state per dt.  M >= N+1. */
MPPI_API int mppi_set_reference(mppi_ctx* ctx, const float* host_ref, int M);

/* Arc-length path P_arc of Alg. 1.  host_pts [P][3]; arc length s_i is the
 * cumulative chord length, the tangent at i is the normalised central difference (periodic when
 * closed != 0, one-sided at the ends otherwise)  [R-22].  2*window+1 <= P <= MPPI_MAX_PATH. */
MPPI_API int mppi_set_path(mppi_ctx* ctx, const float* host_pts, int P, int closed);

/* One MPPI iteration (Alg. 1 lines 3-17) for all B controllers, enqueued on cuda_stream.
 *   d_x0      [B][13] device, in
 *   d_start   [B]     device, in: gate objective: index of the current target gate (wrapped
 *                     mod G); tracking: reference row t0 of the current time (clamped so that
 *                     t0+N <= M-1); contouring: path index hint for the windowed search, or -1
 *                     for a global nearest-vertex search
 *   d_u_nom   [B][N][4] device, in: nominal thrust sequence U*
 *   seed, iter  Philox key and counter word 2
 *   d_u_new   [B][N][4] device, out; may equal d_u_nom exactly (in-place warm start); a partial
 *                     overlap is rejected with MPPI_E_RANGE
 *   d_cost    [B][K] device, out: trajectory costs J_k
 *   d_weights [B][K] device, out: w_k of eq.(4), summing to 1 per controller
 * Outputs are valid once the stream has reached the end of the enqueued work. */
MPPI_API int mppi_step(mppi_ctx* ctx, const float* d_x0, const int32_t* d_start, const float* d_u_nom,
              uint64_t seed, uint32_t iter, float* d_u_new, float* d_cost, float* d_weights,
              void* cuda_stream);

/* n_iters warm-started iterations at a fixed x0 (BASELINE.json configs[1]; [R-14]: no shift):
 * iteration i uses counter word iter0+i and the nominal left by iteration i-1.  d_u [B][N][4] is
 * updated in place; d_cost / d_weights hold the last iteration's values.  With use_graph the
 * whole chain is one graph launch. */
MPPI_API int mppi_optimize(mppi_ctx* ctx, const float* d_x0, const int32_t* d_start, float* d_u,
                  uint64_t seed, uint32_t iter0, int n_iters, float* d_cost, float* d_weights,
                  void* cuda_stream);

/* Same as mppi_step with HOST buffers; returns when the outputs are in the caller's buffers.
 * This is the end-to-end call a host-side control loop makes every cycle.  Fused pipeline: the
 * inputs go down as ONE packed copy from pinned staging memory, the kernel writes u_new (and cost /
 * weights when non-NULL) into mapped host memory itself and raises a sequence number the calling
 * thread polls -- no copy back and no stream synchronisation (a failed stream is still reported:
 * the poll checks cudaStreamQuery every few thousand spins).  Two-pass pipeline, or no mapped
 * memory: explicit copies both ways and cudaStreamSynchronize. */
MPPI_API int mppi_step_host(mppi_ctx* ctx, const float* h_x0, const int32_t* h_start, const float* h_u_nom,
                   uint64_t seed, uint32_t iter, float* h_u_new, float* h_cost, float* h_weights,
                   void* cuda_stream);

/* Closed-loop glue of BASELINE.json configs[4] (receding horizon): the plant
 * (the same RK4 model) applies u_new[b][0] to d_x in place; d_start advances (gate objectives: on a valid
 * pass of the plant segment through the current gate; tracking: +1 row; contouring: windowed
 * nearest vertex); d_u_nom_next[b][t] = d_u_new[b][min(t+1, N-1)].  d_u_nom_next may equal
 * d_u_new. */
MPPI_API int mppi_sim_step(mppi_ctx* ctx, float* d_x, int32_t* d_start, const float* d_u_new,
                  float* d_u_nom_next, void* cuda_stream);

/* MPPI_OBJ_GATE_PAPER: flags of the previous control iteration for the temporal gate-switching check
 * (Fig. 2).  d_prev_front [B][N+1] int32 device, caller-owned, read by every
 * later mppi_step until replaced: entry [b][k] != 0 says that state k of the previous iteration's
 * horizon was in front of the controller's start gate.  A geometric pass of the START gate at state
 * k registers (bonus, target switch) only if that entry is set; passes of later gates of the horizon
 * register on geometry alone.  NULL (the initial setting) = all set = purely geometric.  How the
 * indices of two iterations correspond (same index, or shifted by the control steps elapsed) is the
 * caller's choice: shift the array accordingly. */
MPPI_API int mppi_set_prev_front(mppi_ctx* ctx, const int32_t* d_prev_front);

/* The flags mppi_set_prev_front takes, computed for a nominal sequence: rolls d_u [B][N][4] out from
 * d_x0 [B][13] without noise (thrusts clamped) and writes d_front_out [B][N+1] int32:
 * [b][k] = 1 iff n.(p_k - c) < 0 for the gate d_start[b] (wrapped mod G).  Needs mppi_set_gates. */
MPPI_API int mppi_front_flags(mppi_ctx* ctx, const float* d_x0, const int32_t* d_start, const float* d_u,
                     int32_t* d_front_out, void* cuda_stream);

/* MPPI_OBJ_CONTOUR_PAPER: the fifth column of the nominal and of the update.  d_v_nom [B][N] device, in:
 * nominal progress accelerations; d_v_new [B][N] device, out: v_nom + sum_k w_k dv_k (eq.(5)); the two
 * may be the same buffer (in-place warm start).  Caller-owned, used by every later mppi_step (the fused
 * update writes this column in the same launch) until replaced.  Required before the first step.
 * mppi_optimize needs the in-place form; mppi_step_host and mppi_sim_step return MPPI_E_PARAM under
 * this objective (the plant step is mppi_sim_step_progress). */
MPPI_API int mppi_set_progress(mppi_ctx* ctx, const float* d_v_nom, float* d_v_new);

/* Closed-loop glue under MPPI_OBJ_CONTOUR_PAPER (reading R-39 of DESIGN.md; the counterpart of
 * mppi_sim_step for rows of 19): d_x [B][19] device, in/out: the drone part takes one rate-model RK4 step
 * with d_u_new[b][0] (clamped to the rate range), theta and v_theta advance with d_v_new[b][0] held over
 * the step (theta += dt v_theta + dt^2/2 dv; v_theta clamped to [0, v_theta_max]); d_u_nom_next [B][N][4]
 * and d_v_nom_next [B][N] receive the nominals shifted by one step, last entry repeated.  Each output
 * may be the same buffer as its input (partial overlap: MPPI_E_RANGE).  The start indices are not used
 * by this objective.  One kernel launch on `stream`. */
MPPI_API int mppi_sim_step_progress(mppi_ctx* ctx, float* d_x, const float* d_u_new, float* d_u_nom_next,
                                    const float* d_v_new, float* d_v_nom_next, void* stream);

/* Device pointer to dU [B][N][K][4] of the last step (parity debugging); NULL unless the
 * context keeps it (TWO_PASS pipeline or store_noise). */
MPPI_API const float* mppi_debug_noise(mppi_ctx* ctx);

/* Static facts about the compiled kernels and the launch configuration of this context. */
typedef struct {
    uint32_t struct_size;
    int32_t block_threads, grid_blocks, blocks_per_controller;
    int32_t regs_per_thread, static_smem_bytes, dynamic_smem_bytes, local_bytes_per_thread;
    int32_t max_blocks_per_sm, sm_count;
    int32_t kernels_per_step; /* launches one mppi_step enqueues */
    int32_t samples_per_thread; /* 2 for the packed fp32x2 rollout kernel, else 1 */
    int32_t rollout_warps_per_block; /* latency variant: consumer warps C; pipelined: 3 (5 under input_model 1);
                                        time-parallel: 16 (lanes per rollout); else block_threads / 32 */
    int32_t l2_bytes;
    int64_t scratch_bytes;    /* device memory the context owns */
} mppi_info;
MPPI_API int mppi_get_info(mppi_ctx* ctx, mppi_info* out);

/* Number of kernel launches this context has enqueued since creation. */
MPPI_API int64_t mppi_launch_count(mppi_ctx* ctx);

MPPI_API const char* mppi_error_string(int status);    /* static text for a status code              */
MPPI_API const char* mppi_last_error(mppi_ctx* ctx);   /* detail of the last failure (NULL: of the last
                                                 failed mppi_create / mppi_default_params)  */

/* Roofline denominators measured on the device in use (bench.py).
 * mppi_measure_fma_peak: dependent-chain-free FFMA loop on every SM; writes achieved TFLOP/s.
 * mppi_measure_copy_bw:  device-to-device copy of `bytes`; writes read+write GB/s.
 * Both synchronise and return the best of `reps` timings by CUDA events. */
MPPI_API int mppi_measure_fma_peak(int reps, double* tflops, double* sm_clock_mhz);
MPPI_API int mppi_measure_copy_bw(int64_t bytes, int reps, double* gbs);

/* Issue rates of the instruction classes the rollout loop consists of, for the ceiling of its instruction mix
 * (DESIGN.md section 7): cycles per warp-instruction per SM sub-partition at saturation, measured with clock64.
 * cycles_per_instr [n >= 8], host, out: 0 FFMA with three distinct register operands, 1 FFMA with a constant-bank
 * operand, 2 FFMA2 (packed fp32x2, three register pairs), 3 FMUL, 4 FADD, 5 one Philox half-round (32x32->64
 * multiply + three-input xor: two instructions), 6 MUFU.EX2, 7 FMNMX.  MPPI_E_RANGE if n < 8.  Synchronises. */
MPPI_API int mppi_measure_issue_rates(double* cycles_per_instr, int n);

/* Median time, in microseconds, between two CUDA events that bracket an EMPTY kernel of 128 blocks x 256 threads
 * launched behind a busy GPU (reps launches, 8..4096): the part of any event-timed iteration latency that is the
 * launch and the events, not the library.  Synchronises. */
MPPI_API int mppi_measure_launch_floor(int reps, double* median_us);

/* ---- one entry point that allocates nothing -----------------------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that forbid
 * it): ONE MPPI iteration (Alg. 1 lines 3-17; eq.(3)-(6)) exactly as mppi_create + mppi_set_gates +
 * mppi_step compute it, for the gate-progress objective (MPPI_OBJ_GATE) with rotor-thrust inputs, through the
 * pipelined latency kernel -- with every byte of scratch (block partials, their (m, Z) headers, last-block tickets, the
 * packed gate table) in one file-scope static __device__ array of about 1.07 MB, which every GPU that loads the
 * library holds until the process exits.  No context, no cudaMalloc / cudaFree / cudaHostAlloc, no allocating library
 * routine, on any call.  Limits: K <= MPPI_STATIC_MAX_K, N <= MPPI_STATIC_MAX_N, B <= MPPI_STATIC_MAX_B,
 * G <= MPPI_STATIC_MAX_GATES; beyond them MPPI_E_RANGE, text from mppi_step_static_error().
 *   p          host: parameters as for mppi_create; objective MPPI_OBJ_GATE, input_model 0, pipeline FUSED, store_noise 0,
 *              block_threads 0, variant AUTO or PIPELINED (else MPPI_E_PARAM); fast_math honoured
 *   d_gates    [G][11] DEVICE, in: the rows mppi_set_gates takes (centre, unit normal, unit in-plane axis, half-width,
 *              half-height), not validated here; packed on the device by a one-block kernel in every call
 *   d_x0 [B][13], d_start [B], d_u_nom [B][N][4], d_u_new [B][N][4] (== d_u_nom allowed), d_cost [B][K],
 *   d_weights [B][K]: device, as for mppi_step; seed, iter: Philox key and counter word 2
 * Two kernels are enqueued on cuda_stream; outputs are valid once the stream has reached the end of that work.
 * The first call on a device takes the array's address (cudaGetSymbolAddress) and raises the kernels' dynamic
 * shared-memory limit (cudaFuncSetAttribute) with that device current; a caller that captures graphs makes one plain
 * call first.  Every call shares the one array per device: it keeps the last call's contents (the tickets, which must
 * start at zero, are cleared by every call), and calls that OVERLAP on the GPU -- different streams without an event
 * dependency, concurrent graph replays -- race on it and give wrong results.  Results equal those of the
 * allocating path for the same inputs. */
#define MPPI_STATIC_MAX_K 8192
#define MPPI_STATIC_MAX_N 64
#define MPPI_STATIC_MAX_B 4
#define MPPI_STATIC_MAX_GATES 64
MPPI_API int mppi_step_static(const mppi_params* p, const float* d_gates, int G, const float* d_x0, const int32_t* d_start,
                              const float* d_u_nom, uint64_t seed, uint32_t iter, float* d_u_new, float* d_cost,
                              float* d_weights, void* cuda_stream);
MPPI_API const char* mppi_step_static_error(void); /* detail of this thread's last failed mppi_step_static ("" if none) */

#ifdef __cplusplus
}
#endif
#endif /* MPPI_H_ */
