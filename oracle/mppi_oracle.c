/*
 * mppi_oracle.c -- float64 CPU oracle for one MPPI iteration of the reference-free racing
 * controller of arXiv 2509.14726.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
 * source, header, table or helper with the CUDA path under paper_2509_14726_b200/csrc/.
 *
 * It is the algorithm written out step by step in the paper's order (Alg. 1),
 * all arithmetic in double, all integer work exact, nothing blocked, fused or reordered beyond
 * what the cited passage states.  The only parallelism is OpenMP over the independent samples
 * ("for m = 1 to M", Alg. 1 line 5).  Citations are PAPER.md:<line> plus the
 * section / equation, or a reading [R-n] listed in DESIGN.md (taken from SURVEY.md section 8(c)).
 *
 * Notation: the paper writes M samples and K horizon steps; BASELINE.json writes
 * K samples and N horizon steps.  This file uses K samples, N steps, B independent controllers.
 *
 * Pins (tests/test_oracle_*.py, run with -m "not gpu"): Philox known-answer vectors; hover
 * invariant; closed-form free fall; yaw / roll / pitch torque closed forms; torque-free
 * precession; quaternion norm; hand-built gate cases; softmax invariants; a K=1,N=1 step by
 * hand; the survey's worked example (tests/golden/); an independently written numpy evaluator.
 * The paper's own J_gate (objective 3) and input model (input_model = 1) have their own pins in
 * tests/test_oracle_gate_paper.py and tests/test_oracle_rate_model.py (hand-built segments, free-fall
 * flags, thrust-ramp / torque / drag closed forms, the numpy evaluator's own branches).
 * "parity unpinned": the numbers of the five BASELINE.json configs themselves -- the paper
 * prints no hot-path values -- and the uniform->normal mapping beyond its moments (it is a
 * definition, [R-2],[R-3]).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_OBJ_GATE 0
#define ORC_OBJ_TRACK 1
#define ORC_OBJ_CONTOUR 2
#define ORC_OBJ_CONTOUR_PAPER 4 /* the paper's own J_contour: theta, v_theta states, Delta v_theta sampled, eq.(9) */
#define ORC_OBJ_GATE_PAPER 3   /* the paper's own J_gate, eq.(6),(7) + temporal check */

typedef struct {
    int32_t K, N, B, objective;
    double dt, lambda, sigma;
    double mass, Jx, Jy, Jz, arm, c_tau, g;
    double T_min, T_max;
    double w_omega;
    double gate_miss_penalty, gate_pass_bonus;
    double Qp, Qv, Qq, Qw, R;
    double q_contour, q_lag, mu_progress;
    int32_t window;
    int32_t near_mode;       /* eq.(7): which gate the near term measures against: 0 = the step's own target [R-24],
                                1 = the horizon's start gate p0_gate, before and after the switch [R-40]        */
    double q_near, r_near;   /* eq.(7): weight and threshold radius [R-24] */
    /* the paper's own input model, PAPER.md:72 and Table I */
    int32_t input_model;     /* 0: rotor thrusts are the inputs (configs); 1: u = dT/dt, thrusts are states */
    int32_t pad2_;
    double rate_max;         /* |u_i| <= rate_max, N/s (Table I "Delta T_s [-10,10]") [R-28]            */
    double drag_x, drag_y, drag_z; /* D = diag(.) of eq.(2), body frame, 1/s [R-30]                       */
    double w_limit, omega_max;     /* "external cost" on the body-rate range [R-31]         */
    /* the paper's own contouring formulation, eq.(9), Table I */
    double sigma_v;          /* std of the sampled progress acceleration Delta v_theta, m/s^2 [R-35]     */
    double dv_max;           /* |Delta v_theta| <= dv_max (Table I "[-20,20]")                           */
    double v_theta_max;      /* 0 <= v_theta <= v_theta_max (eq.(9); Table I "[0,10]")                   */
    double r_dv;             /* weight of |Delta v_theta|^2                                              */
} orc_params;

typedef struct {
    int32_t G;           /* gates            */
    int32_t M;           /* reference rows   */
    int32_t P;           /* path points      */
    int32_t closed;      /* path is periodic */
    const double* gates; /* [G][11]: centre c(3), unit normal n(3) = direction of travel,
                            unit in-plane axis h(3), half-width along h, half-height along v=h x n */
    const double* ref;   /* [M][13]: p(3), q wxyz(4), v(3), omega(3) */
    const double* pts;   /* [P][3]  */
    /* ORC_OBJ_CONTOUR_PAPER: the fifth column of the nominal and of the update [R-35] */
    const double* v_nom;  /* [B][N]  nominal progress accelerations                     (in)          */
    double* v_new;        /* [B][N]  updated ones, eq.(5) applied to the fifth input     (out)         */
    double* dv_out;       /* [B][K][N] or NULL: the clamped perturbations actually applied (out)       */
    const int32_t* prev_front; /* [B][N+1] or NULL: ORC_OBJ_GATE_PAPER, state k of the previous control
                            iteration was in front of the start gate (Fig. 2) [R-25] */
} orc_track;

/* ------------------------------------------------------------------------------------------
 * Philox4x32-10 (Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3",
 * SC'11).  [R-1]: the paper only asks for independent Gaussian perturbations (eq.(3),
 * PAPER.md:78-82); BASELINE.json:north_star fixes "a counter-based Philox stream keyed by
 * (seed, iter, sample, step)".  counter = (sample k, step t, iter, controller b),
 * key = (seed low word, seed high word).
 * ---------------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = M0 * (uint64_t)c0;
        uint64_t p1 = M1 * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        c0 = hi1 ^ c1 ^ k0;
        c1 = lo1;
        c2 = hi0 ^ c3 ^ k1;
        c3 = lo0;
        k0 += W0; /* the key is bumped between rounds (applied before the next one) */
        k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* [R-2] uint32 -> uniform on the open interval: u = (2 (r >> 9) + 1) * 2^-24.  The 23-bit
 * lattice is exact in fp32 and fp64 and never reaches 0 or 1. */
double orc_uniform(uint32_t r)
{
    return (double)(2u * (r >> 9) + 1u) * (1.0 / 16777216.0);
}

/* [R-3] basic Box-Muller: words (r0,r1) -> rotors 0,1 (cos, sin); (r2,r3) -> rotors 2,3.
 * Realises delta u ~ N(0, Sigma), Sigma = sigma^2 I (eq.(3)). */
void orc_normals(uint64_t seed, uint32_t k, uint32_t t, uint32_t iter, uint32_t b, double z[4])
{
    const double two_pi = 6.283185307179586476925286766559;
    uint32_t ctr[4] = { k, t, iter, b };
    uint32_t key[2] = { (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32) };
    uint32_t r[4];
    orc_philox4x32_10(ctr, key, r);
    double rad0 = sqrt(-2.0 * log(orc_uniform(r[0])));
    double rad1 = sqrt(-2.0 * log(orc_uniform(r[2])));
    z[0] = rad0 * cos(two_pi * orc_uniform(r[1]));
    z[1] = rad0 * sin(two_pi * orc_uniform(r[1]));
    z[2] = rad1 * cos(two_pi * orc_uniform(r[3]));
    z[3] = rad1 * sin(two_pi * orc_uniform(r[3]));
}

/* ------------------------------------------------------------------------------------------
 * Quadrotor rigid-body dynamics f_dyn, eq.(2), thrust/torque map PAPER.md:70.
 * State order (BASELINE.json configs[0]): x = [p(3), q(w,x,y,z), v(3), omega(3)].
 * [R-6] torque signs literal; body z is the thrust axis; world z up, gravity (0,0,-g).
 * [R-7] rotor drag D = 0 (no value anywhere in the paper).  [D-1] input = rotor thrusts.
 * ---------------------------------------------------------------------------------------- */
void orc_fdyn(const orc_params* P, const double x[13], const double T[4], double xd[13])
{
    const double qw = x[3], qx = x[4], qy = x[5], qz = x[6];
    const double vx = x[7], vy = x[8], vz = x[9];
    const double ox = x[10], oy = x[11], oz = x[12];

    /* p_dot = v */
    xd[0] = vx; xd[1] = vy; xd[2] = vz;

    /* q_dot = 1/2 Lambda(q) [0; omega]  = 1/2 q (x) (0, omega), omega in the body frame */
    xd[3] = 0.5 * (-qx * ox - qy * oy - qz * oz);
    xd[4] = 0.5 * ( qw * ox + qy * oz - qz * oy);
    xd[5] = 0.5 * ( qw * oy + qz * ox - qx * oz);
    xd[6] = 0.5 * ( qw * oz + qx * oy - qy * ox);

    /* v_dot = g + (1/m) R(q) T,  T = [0, 0, sum T_s]: third column of R(q) */
    const double S = T[0] + T[1] + T[2] + T[3];
    const double r13 = 2.0 * (qx * qz + qw * qy);
    const double r23 = 2.0 * (qy * qz - qw * qx);
    const double r33 = 1.0 - 2.0 * (qx * qx + qy * qy);
    xd[7] = (S / P->mass) * r13;
    xd[8] = (S / P->mass) * r23;
    xd[9] = (S / P->mass) * r33 - P->g;
    if (P->drag_x != 0.0 || P->drag_y != 0.0 || P->drag_z != 0.0) {
        /* - R D R^T v, D = diag(drag) in the body frame (eq.(2)) [R-30]: full R(q) */
        const double R[3][3] = {
            { 1.0 - 2.0 * (qy * qy + qz * qz), 2.0 * (qx * qy - qw * qz), r13 },
            { 2.0 * (qx * qy + qw * qz), 1.0 - 2.0 * (qx * qx + qz * qz), r23 },
            { 2.0 * (qx * qz - qw * qy), 2.0 * (qy * qz + qw * qx), r33 } };
        const double d[3] = { P->drag_x, P->drag_y, P->drag_z };
        const double v[3] = { vx, vy, vz };
        for (int j = 0; j < 3; ++j) {                      /* body axis j = column j of R */
            const double vb = R[0][j] * v[0] + R[1][j] * v[1] + R[2][j] * v[2];   /* (R^T v)_j */
            for (int i = 0; i < 3; ++i) xd[7 + i] -= R[i][j] * d[j] * vb;
        }
    }

    /* omega_dot = J^-1 (tau - omega x J omega) */
    const double lever = P->arm / sqrt(2.0);
    const double tx = lever * ( T[0] + T[1] - T[2] - T[3]);
    const double ty = lever * (-T[0] + T[1] + T[2] - T[3]);
    const double tz = P->c_tau * (T[0] - T[1] + T[2] - T[3]);
    const double Lx = P->Jx * ox, Ly = P->Jy * oy, Lz = P->Jz * oz; /* J omega */
    const double cx = oy * Lz - oz * Ly;                             /* omega x J omega */
    const double cy = oz * Lx - ox * Lz;
    const double cz = ox * Ly - oy * Lx;
    xd[10] = (tx - cx) / P->Jx;
    xd[11] = (ty - cy) / P->Jy;
    xd[12] = (tz - cz) / P->Jz;
}

/* Discretisation f ("discrete-time dynamics model with time step dt").
 * [R-4] classical 4-stage Runge-Kutta on the full 13-vector, input held over the step.
 * [R-5] quaternion renormalised once after the full step. */
void orc_rk4_step(const orc_params* P, const double x[13], const double T[4], double dt,
                  double xn[13])
{
    double k1[13], k2[13], k3[13], k4[13], xs[13];
    orc_fdyn(P, x, T, k1);
    for (int i = 0; i < 13; ++i) xs[i] = x[i] + 0.5 * dt * k1[i];
    orc_fdyn(P, xs, T, k2);
    for (int i = 0; i < 13; ++i) xs[i] = x[i] + 0.5 * dt * k2[i];
    orc_fdyn(P, xs, T, k3);
    for (int i = 0; i < 13; ++i) xs[i] = x[i] + dt * k3[i];
    orc_fdyn(P, xs, T, k4);
    for (int i = 0; i < 13; ++i)
        xn[i] = x[i] + (dt / 6.0) * (k1[i] + 2.0 * k2[i] + 2.0 * k3[i] + k4[i]);
    const double nq = sqrt(xn[3] * xn[3] + xn[4] * xn[4] + xn[5] * xn[5] + xn[6] * xn[6]);
    for (int i = 3; i < 7; ++i) xn[i] /= nq;
}

/* The paper's own input model ("Following the approach in [4], we define the control
 * input u as the derivative of the single rotor thrust"): state x = [p, q, v, omega, T(4)] (17),
 * T' = u held over the step [R-27].  Classical RK4 on the 17-vector (the stage thrusts are
 * T, T + dt/2 u, T + dt/2 u, T + dt u, unclamped), quaternion renormalised, then the thrust STATES
 * are projected onto [T_min, T_max] (Table I "T_s [0,10]"; the paper's soft external cost for the
 * range has no printed form) [R-29]. */
void orc_rk4_rate_step(const orc_params* P, const double x[17], const double u[4], double dt,
                       double xn[17])
{
    double k[4][17], xs[17];
    memcpy(xs, x, sizeof xs);
    for (int st = 0; st < 4; ++st) {
        orc_fdyn(P, xs, xs + 13, k[st]);
        for (int i = 0; i < 4; ++i) k[st][13 + i] = u[i];
        if (st == 3) break;
        const double c = st == 2 ? dt : 0.5 * dt;
        for (int i = 0; i < 17; ++i) xs[i] = x[i] + c * k[st][i];
    }
    for (int i = 0; i < 17; ++i)
        xn[i] = x[i] + (dt / 6.0) * (k[0][i] + 2.0 * k[1][i] + 2.0 * k[2][i] + k[3][i]);
    const double nq = sqrt(xn[3] * xn[3] + xn[4] * xn[4] + xn[5] * xn[5] + xn[6] * xn[6]);
    for (int i = 3; i < 7; ++i) xn[i] /= nq;
    for (int i = 13; i < 17; ++i) xn[i] = fmin(fmax(xn[i], P->T_min), P->T_max);
}

/* "External cost" for the body-rate range of Table I [R-31]:
 * w_limit sum_i max(0, |omega_i| - omega_max)^2 on a state's body rates. */
double orc_rate_limit_cost(const orc_params* P, const double omega[3])
{
    double J = 0.0;
    for (int i = 0; i < 3; ++i) {
        const double e = fabs(omega[i]) - P->omega_max;
        if (e > 0.0) J += e * e;
    }
    return P->w_limit * J;
}

/* ------------------------------------------------------------------------------------------
 * Gate-progress step cost.  Progress term of eq.(6) PAPER.md:105-110 with un-squared
 * distances [D-2]; in-horizon target switching PAPER.md:112; the pass is "geometrically
 * defined by the quadrotor flying through the gate" [R-9],[R-10]; constants
 * from BASELINE.json configs[0] (+miss on a crossing outside the opening, -bonus and target
 * switch on a valid crossing, w_omega |omega|^2).
 * Returns the step cost; *gate is advanced on a valid pass (applies from the NEXT step).
 * *margin is lowered to the smallest distance of any discrete decision from its threshold
 * [R-19]; *ncross counts valid passes.
 * ---------------------------------------------------------------------------------------- */
static double dot3(const double a[3], const double b[3])
{
    return a[0] * b[0] + a[1] * b[1] + a[2] * b[2];
}

double orc_gate_step(const orc_params* P, const orc_track* trk, const double p_prev[3],
                     const double p[3], const double omega[3], int32_t* gate, double* margin,
                     int32_t* ncross)
{
    const double* gt = trk->gates + 11 * (*gate);
    const double* c = gt; const double* n = gt + 3; const double* h = gt + 6;
    const double a_h = gt[9], a_v = gt[10];
    const double v[3] = { h[1] * n[2] - h[2] * n[1], h[2] * n[0] - h[0] * n[2],
                          h[0] * n[1] - h[1] * n[0] };           /* v = h x n */
    double r_prev[3], r[3];
    for (int i = 0; i < 3; ++i) { r_prev[i] = p_prev[i] - c[i]; r[i] = p[i] - c[i]; }

    double J = sqrt(dot3(r, r)) - sqrt(dot3(r_prev, r_prev));   /* d_t - d_{t-1} */

    const double s_prev = dot3(n, r_prev), s = dot3(n, r);      /* signed plane distances */
    if (margin) {
        if (fabs(s_prev) < *margin) *margin = fabs(s_prev);
        if (fabs(s) < *margin) *margin = fabs(s);
    }
    if (s_prev < 0.0 && s >= 0.0) {                              /* front -> back crossing */
        const double alpha = s_prev / (s_prev - s);
        double rx[3];
        for (int i = 0; i < 3; ++i) rx[i] = r_prev[i] + alpha * (r[i] - r_prev[i]);
        const double y = dot3(h, rx), z = dot3(v, rx);
        if (margin) {
            if (fabs(fabs(y) - a_h) < *margin) *margin = fabs(fabs(y) - a_h);
            if (fabs(fabs(z) - a_v) < *margin) *margin = fabs(fabs(z) - a_v);
        }
        if (fabs(y) <= a_h && fabs(z) <= a_v) {
            J -= P->gate_pass_bonus;
            *gate = (*gate + 1) % trk->G;
            if (ncross) *ncross += 1;
        } else {
            J += P->gate_miss_penalty;                           /* miss: target unchanged */
        }
    }
    J += P->w_omega * dot3(omega, omega);
    return J;
}

/* ------------------------------------------------------------------------------------------
 * Trajectory-tracking cost, eq.(8) PAPER.md:139-147.  [R-11]: stage terms on the pre-step
 * states k = 0..N-1 paired with the input applied at k, terminal term on state N with
 * Q_K = Q; quaternion error |q - s q_ref|^2, s = sign(q . q_ref) (double cover);
 * R on (T - hover) per BASELINE.json configs[2].
 * ---------------------------------------------------------------------------------------- */
/* ------------------------------------------------------------------------------------------
 * The paper's own gate-progress objective, one step (eq.(6),(7) PAPER.md:105-129), readings
 * [R-23]..[R-25] of DESIGN.md:
 *   progress   |p_{t+1} - c|^2 - |p_t - c|^2, squared distances, against the gate targeted at the
 *              start of the step                                                 (eq.(6))
 *   near term  + Q_near |p_t - c|^2 when |p_t - c| < r_near (pre-step state p_k)  (eq.(7))
 *   switching  a front->back crossing of the target plane inside the opening is REGISTERED (bonus,
 *              target <- next gate from the next step on) only if the target is not the horizon's
 *              start gate, or the corresponding state of the previous control iteration was in
 *              front of the gate: front_ok != 0 (Fig. 2).  An unregistered pass
 *              changes nothing; a crossing outside the opening adds the miss penalty, as in
 *              orc_gate_step.
 *   body rates + w_omega |omega_{t+1}|^2
 * margin additionally tracks | |p_t - c| - r_near | (the near term is discontinuous there).
 * ---------------------------------------------------------------------------------------- */
double orc_gate_paper_step(const orc_params* P, const orc_track* trk, const double p_prev[3],
                           const double p[3], const double omega[3], int32_t* gate, int32_t gate0,
                           int32_t front_ok, double* margin, int32_t* ncross)
{
    const double* gt = trk->gates + 11 * (*gate);
    const double* c = gt; const double* n = gt + 3; const double* h = gt + 6;
    const double a_h = gt[9], a_v = gt[10];
    const double v[3] = { h[1] * n[2] - h[2] * n[1], h[2] * n[0] - h[0] * n[2],
                          h[0] * n[1] - h[1] * n[0] };           /* v = h x n */
    double r_prev[3], r[3];
    for (int i = 0; i < 3; ++i) { r_prev[i] = p_prev[i] - c[i]; r[i] = p[i] - c[i]; }
    const double d2_prev = dot3(r_prev, r_prev), d2 = dot3(r, r);

    double J = d2 - d2_prev;                                     /* eq.(6) */
    /* eq.(7), on the pre-step state p_k.  near_mode 0 [R-24]: against the step's own target gate.
     * near_mode 1 [R-40]: "prevent states near the current gate p0_gate ... from deviating too much from it" read
     * literally -- against the horizon's START gate gate0, also for the states that already target the next gate */
    double dn2 = d2_prev;
    if (P->near_mode == 1 && *gate != gate0) {
        const double* c0 = trk->gates + 11 * gate0;
        double r0[3];
        for (int i = 0; i < 3; ++i) r0[i] = p_prev[i] - c0[i];
        dn2 = dot3(r0, r0);
    }
    const double d_near = sqrt(dn2);
    if (d_near < P->r_near) J += P->q_near * dn2;
    if (margin && fabs(d_near - P->r_near) < *margin) *margin = fabs(d_near - P->r_near);

    const double s_prev = dot3(n, r_prev), s = dot3(n, r);
    if (margin) {
        if (fabs(s_prev) < *margin) *margin = fabs(s_prev);
        if (fabs(s) < *margin) *margin = fabs(s);
    }
    if (s_prev < 0.0 && s >= 0.0) {
        const double alpha = s_prev / (s_prev - s);
        double rx[3];
        for (int i = 0; i < 3; ++i) rx[i] = r_prev[i] + alpha * (r[i] - r_prev[i]);
        const double y = dot3(h, rx), z = dot3(v, rx);
        if (margin) {
            if (fabs(fabs(y) - a_h) < *margin) *margin = fabs(fabs(y) - a_h);
            if (fabs(fabs(z) - a_v) < *margin) *margin = fabs(fabs(z) - a_v);
        }
        if (fabs(y) <= a_h && fabs(z) <= a_v) {
            if (*gate != gate0 || front_ok) {                    /* temporally consistent pass */
                J -= P->gate_pass_bonus;
                *gate = (*gate + 1) % trk->G;
                if (ncross) *ncross += 1;
            }
        } else {
            J += P->gate_miss_penalty;
        }
    }
    J += P->w_omega * dot3(omega, omega);
    return J;
}

/* "In front of the gate" flags of a nominal rollout [R-26]: front[k] = 1 iff n.(p_k - c) < 0 for the
 * start gate, k = 0..N, states of the noise-free rollout of u (clamped) from x0.  margin (may be
 * NULL) receives min_k |n.(p_k - c)|. */
void orc_front_flags(const orc_params* P, const orc_track* trk, const double x0[13], int32_t start,
                     const double* u /*[N][4]*/, int32_t* front /*[N+1]*/, double* margin)
{
    int32_t g = start % trk->G; if (g < 0) g += trk->G;
    const double* c = trk->gates + 11 * g; const double* n = c + 3;
    const int rate = P->input_model == 1;                    /* x0 then has 17 entries, u are rates */
    double x[17], xn[17], mg = INFINITY;
    memcpy(x, x0, sizeof(double) * (rate ? 17 : 13));
    for (int k = 0; k <= P->N; ++k) {
        const double r[3] = { x[0] - c[0], x[1] - c[1], x[2] - c[2] };
        const double s = dot3(n, r);
        front[k] = s < 0.0 ? 1 : 0;
        if (fabs(s) < mg) mg = fabs(s);
        if (k == P->N) break;
        double T[4];
        const double lo = rate ? -P->rate_max : P->T_min, hi = rate ? P->rate_max : P->T_max;
        for (int i = 0; i < 4; ++i) T[i] = fmin(fmax(u[4 * k + i], lo), hi);
        if (rate) orc_rk4_rate_step(P, x, T, P->dt, xn);
        else orc_rk4_step(P, x, T, P->dt, xn);
        memcpy(x, xn, sizeof(double) * (rate ? 17 : 13));
    }
    if (margin) *margin = mg;
}

double orc_track_state_term(const orc_params* P, const double x[13], const double xr[13])
{
    double ep = 0, eq = 0, ev = 0, ew = 0;
    for (int i = 0; i < 3; ++i) { double d = x[i] - xr[i]; ep += d * d; }
    double qdot = x[3] * xr[3] + x[4] * xr[4] + x[5] * xr[5] + x[6] * xr[6];
    const double s = (qdot < 0.0) ? -1.0 : 1.0;
    for (int i = 3; i < 7; ++i) { double d = x[i] - s * xr[i]; eq += d * d; }
    for (int i = 7; i < 10; ++i) { double d = x[i] - xr[i]; ev += d * d; }
    for (int i = 10; i < 13; ++i) { double d = x[i] - xr[i]; ew += d * d; }
    return P->Qp * ep + P->Qv * ev + P->Qq * eq + P->Qw * ew;
}

double orc_track_stage(const orc_params* P, const double x[13], const double T[4],
                       const double xr[13])
{
    const double hover = P->mass * P->g / 4.0;
    double eu = 0;
    for (int i = 0; i < 4; ++i) { double d = T[i] - hover; eu += d * d; }
    return orc_track_state_term(P, x, xr) + P->R * eu;
}

/* ------------------------------------------------------------------------------------------
 * Arc-length path helpers.  "converted into an arc-length parameterized representation"
 * (PAPER.md:239).  [R-22]: s_0 = 0, s_i = s_{i-1} + |P_i - P_{i-1}| (cumulative chord
 * length); closed length L = s_{P-1} + |P_0 - P_{P-1}|; tangent t_i = unit(P_{i+1} - P_{i-1})
 * with periodic neighbours when closed, one-sided differences at the two ends when open.
 * s[P], tan[P][3] are written; returns L (closed) or s_{P-1} (open).
 * ---------------------------------------------------------------------------------------- */
double orc_path_prepare(const double* pts, int32_t Pn, int32_t closed, double* s, double* tan)
{
    s[0] = 0.0;
    for (int i = 1; i < Pn; ++i) {
        double d[3];
        for (int a = 0; a < 3; ++a) d[a] = pts[3 * i + a] - pts[3 * (i - 1) + a];
        s[i] = s[i - 1] + sqrt(dot3(d, d));
    }
    double L = s[Pn - 1];
    if (closed) {
        double d[3];
        for (int a = 0; a < 3; ++a) d[a] = pts[a] - pts[3 * (Pn - 1) + a];
        L += sqrt(dot3(d, d));
    }
    for (int i = 0; i < Pn; ++i) {
        int ip = i + 1, im = i - 1;
        if (closed) { ip = ip % Pn; im = (im + Pn) % Pn; }
        else { if (ip > Pn - 1) ip = Pn - 1; if (im < 0) im = 0; }
        double d[3];
        for (int a = 0; a < 3; ++a) d[a] = pts[3 * ip + a] - pts[3 * im + a];
        const double nd = sqrt(dot3(d, d));
        for (int a = 0; a < 3; ++a) tan[3 * i + a] = d[a] / nd;
    }
    return L;
}

/* Nearest path vertex to p among offsets -W..+W around `centre`, scanned in increasing offset,
 * first minimiser wins [R-12]; centre < 0 means a global scan i = 0..P-1.  Open paths skip
 * indices outside [0, P-1]. */
int32_t orc_path_nearest(const double* pts, int32_t Pn, int32_t closed, const double p[3],
                         int32_t centre, int32_t W)
{
    double best = INFINITY; int32_t ibest = -1;
    int lo = centre - W, hi = centre + W;
    if (centre < 0) { lo = 0; hi = Pn - 1; }
    for (int j = lo; j <= hi; ++j) {
        int i = j;
        if (closed) i = ((j % Pn) + Pn) % Pn;
        else if (i < 0 || i >= Pn) continue;
        double d[3];
        for (int a = 0; a < 3; ++a) d[a] = p[a] - pts[3 * i + a];
        const double d2 = dot3(d, d);
        if (d2 < best) { best = d2; ibest = i; }
    }
    return ibest;
}

/* Projection onto the tangent line at vertex i: lag error e_l (tangential), contouring error
 * squared e_c^2 (perpendicular), progress theta = s_i + e_l  ([R-12],[R-13]). */
static void orc_path_project(const double* pts, const double* s, const double* tan, int32_t i,
                             const double p[3], double* e_l, double* e_c2, double* theta)
{
    double e[3];
    for (int a = 0; a < 3; ++a) e[a] = p[a] - pts[3 * i + a];
    *e_l = dot3(e, tan + 3 * i);
    double c2 = dot3(e, e) - (*e_l) * (*e_l);
    *e_c2 = c2 > 0.0 ? c2 : 0.0;
    *theta = s[i] + *e_l;
}

/* Contouring step cost, eq.(9) PAPER.md:149-161 in the projection variant of
 * BASELINE.json configs[3] [D-6]: q_c e_c^2 + q_l e_l^2 - mu (theta - theta_prev)
 * + w_omega |omega|^2; idx and theta_prev are carried along the rollout. */
double orc_contour_step(const orc_params* P, const orc_track* trk, const double* s,
                        const double* tan, double L, const double p[3], const double omega[3],
                        int32_t* idx, double* theta_prev)
{
    const int32_t i = orc_path_nearest(trk->pts, trk->P, trk->closed, p, *idx, P->window);
    double e_l, e_c2, theta;
    orc_path_project(trk->pts, s, tan, i, p, &e_l, &e_c2, &theta);
    double d = theta - *theta_prev;
    if (trk->closed) {                       /* wrap into (-L/2, L/2] */
        while (d > 0.5 * L) d -= L;
        while (d <= -0.5 * L) d += L;
    }
    *idx = i; *theta_prev = theta;
    return P->q_contour * e_c2 + P->q_lag * e_l * e_l - P->mu_progress * d
         + P->w_omega * dot3(omega, omega);
}

/* ------------------------------------------------------------------------------------------
 * The paper's own contouring formulation, eq.(9): the progress
 * theta and its speed v_theta are STATES, the progress acceleration Delta v_theta is a fifth sampled
 * input next to the four thrust rates Delta T (so it needs input_model = 1), and the path is looked
 * up BY theta instead of searched.  Readings [R-33]..[R-37] of DESIGN.md.
 * ---------------------------------------------------------------------------------------- */
/* P(theta) and the unit tangent at theta [R-36]: theta wrapped into [0, L) on a closed path (clamped
 * to [0, s_last] on an open one); segment i with s_i <= theta < s_{i+1} (the closing segment runs from
 * the last point to the first, s_P = L); linear interpolation of the points, normalised linear
 * interpolation of the vertex tangents of [R-22]. */
void orc_path_eval(const double* pts, const double* s, const double* tan, int32_t Pn, int32_t closed,
                   double L, double theta, double pos[3], double tg[3])
{
    double th = theta;
    if (closed) { th = fmod(th, L); if (th < 0.0) th += L; }
    else { if (th < 0.0) th = 0.0; if (th > s[Pn - 1]) th = s[Pn - 1]; }
    int i = 0;
    const int last = closed ? Pn - 1 : Pn - 2;
    while (i < last && s[i + 1] <= th) ++i;
    const int j = (i + 1) % Pn;
    const double s1 = (i + 1 < Pn) ? s[i + 1] : L;
    double lam = (th - s[i]) / (s1 - s[i]);
    if (lam > 1.0) lam = 1.0;
    double t[3];
    for (int a = 0; a < 3; ++a) {
        pos[a] = (1.0 - lam) * pts[3 * i + a] + lam * pts[3 * j + a];
        t[a] = (1.0 - lam) * tan[3 * i + a] + lam * tan[3 * j + a];
    }
    const double nt = sqrt(dot3(t, t));
    for (int a = 0; a < 3; ++a) tg[a] = t[a] / nt;
}

/* the fifth standard normal of a (sample, step): first Box-Muller output of Philox4x32-10 at counter
 * (k, t + 2^31, iter, b), same key -- a block the four rotor normals never use [R-35] */
double orc_normal5(uint64_t seed, uint32_t k, uint32_t t, uint32_t iter, uint32_t b)
{
    double z[4];
    orc_normals(seed, k, t + 0x80000000u, iter, b, z);
    return z[0];
}

/* stage cost of eq.(9) at a pre-step state [R-37] */
double orc_contour_paper_stage(const orc_params* P, const orc_track* trk, const double* s, const double* tan,
                               double L, const double x[19], const double dT[4], double dv)
{
    double pos[3], tg[3];
    orc_path_eval(trk->pts, s, tan, trk->P, trk->closed, L, x[17], pos, tg);
    const double e[3] = { x[0] - pos[0], x[1] - pos[1], x[2] - pos[2] };
    const double e_l = dot3(e, tg);
    double e_c2 = dot3(e, e) - e_l * e_l;
    if (e_c2 < 0.0) e_c2 = 0.0;
    double r = 0.0;
    for (int i = 0; i < 4; ++i) r += dT[i] * dT[i];
    return P->q_lag * e_l * e_l + P->q_contour * e_c2 + P->w_omega * dot3(x + 10, x + 10)
         + P->r_dv * dv * dv + P->R * r - P->mu_progress * x[18];
}

/* progress states over one step with the acceleration held [R-34] */
void orc_progress_step(const orc_params* P, double theta, double v, double dv, double* theta_n, double* v_n)
{
    *theta_n = theta + P->dt * v + 0.5 * P->dt * P->dt * dv;
    *v_n = fmin(fmax(v + P->dt * dv, 0.0), P->v_theta_max);
}

/* ------------------------------------------------------------------------------------------
 * One sample: Alg. 1 lines 6-13.  Writes du[N][4] (the clamped
 * perturbation actually rolled out [R-8]) and returns the trajectory cost J.
 * ---------------------------------------------------------------------------------------- */
typedef struct { const double* s; const double* tan; double L; } orc_path_aux;

double orc_rollout_cost(const orc_params* P, const orc_track* trk, const orc_path_aux* pa,
                        const double* x0 /*[13 | 17 | 19]*/, int32_t start, const double* u_nom /*[N][4]*/,
                        uint64_t seed, uint32_t iter, uint32_t k, uint32_t b,
                        double* du /*[N][4]*/, double* margin, int32_t* ncross, int32_t* aux_end,
                        double* x_end /*[13] or NULL*/)
{
    const int rate = P->input_model == 1;            /* x0 then has 17 entries: ..., T(4) */
    const int cpaper = P->objective == ORC_OBJ_CONTOUR_PAPER;   /* ... and theta, v_theta: 19 [R-33] */
    const int xdim = cpaper ? 19 : (rate ? 17 : 13);
    double x[19];
    memcpy(x, x0, sizeof(double) * xdim);
    if (P->objective == ORC_OBJ_TRACK) {
        /* [R-11] the reference row of the current time is clamped so that the horizon's last row start + N
         * exists (include/mppi.h, mppi_step: "clamped so that t0+N <= M-1"): the clock stops at the end of
         * the reference, as in orc_sim_step */
        if (start > trk->M - 1 - P->N) start = trk->M - 1 - P->N;
        if (start < 0) start = 0;
    }
    int32_t aux = start;
    if (P->objective == ORC_OBJ_GATE_PAPER || P->objective == ORC_OBJ_GATE) {   /* target index wraps mod G [R-10] */
        aux = start % trk->G;
        if (aux < 0) aux += trk->G;
    }
    const int32_t gate0 = aux;
    double J = 0.0, theta_prev = 0.0;
    double marg = INFINITY; int32_t nc = 0;

    if (P->objective == ORC_OBJ_CONTOUR) {
        /* initial index: windowed search around the hint, or global when the hint is -1;
         * theta_prev from p_0 with the same projection formula [R-13] */
        double e_l, e_c2;
        aux = orc_path_nearest(trk->pts, trk->P, trk->closed, x, start, P->window);
        orc_path_project(trk->pts, pa->s, pa->tan, aux, x, &e_l, &e_c2, &theta_prev);
    }

    for (int t = 0; t < P->N; ++t) {
        double z[4], T[4];
        orc_normals(seed, k, (uint32_t)t, iter, b, z);                   /* eq.(3) */
        const double lo = rate ? -P->rate_max : P->T_min, hi = rate ? P->rate_max : P->T_max;
        for (int i = 0; i < 4; ++i) {
            double Ti = u_nom[4 * t + i] + P->sigma * z[i];
            Ti = fmin(fmax(Ti, lo), hi);          /* hard clamp [D-5]; thrust rates: [R-28] */
            T[i] = Ti;
            du[4 * t + i] = Ti - u_nom[4 * t + i];                         /* [R-8] */
        }
        if (P->objective == ORC_OBJ_TRACK) {
            if (rate) {                           /* eq.(8): ||u_k||^2_R on the inputs = the rates [R-32] */
                double eu = 0.0;
                for (int i = 0; i < 4; ++i) eu += T[i] * T[i];
                J += orc_track_state_term(P, x, trk->ref + 13 * (start + t)) + P->R * eu;
            } else {
                J += orc_track_stage(P, x, T, trk->ref + 13 * (start + t));    /* eq.(8) stage */
            }
        }

        double dv = 0.0;
        if (cpaper) {                             /* fifth sampled input + stage cost of eq.(9) [R-35],[R-37] */
            const double vn = trk->v_nom[(size_t)b * P->N + t];
            dv = fmin(fmax(vn + P->sigma_v * orc_normal5(seed, k, (uint32_t)t, iter, b), -P->dv_max), P->dv_max);
            if (trk->dv_out) trk->dv_out[((size_t)b * P->K + k) * P->N + t] = dv - vn;
            J += orc_contour_paper_stage(P, trk, pa->s, pa->tan, pa->L, x, T, dv);
        }

        double xn[19];
        if (cpaper) orc_progress_step(P, x[17], x[18], dv, &xn[17], &xn[18]);   /* [R-34] */
        if (rate) orc_rk4_rate_step(P, x, T, P->dt, xn);                   /* [R-27],[R-29] */
        else orc_rk4_step(P, x, T, P->dt, xn);                             /* Alg.1 l.7-9 */
        if (rate) J += orc_rate_limit_cost(P, xn + 10);                    /* [R-31] */

        if (P->objective == ORC_OBJ_GATE)
            J += orc_gate_step(P, trk, x, xn, xn + 10, &aux, &marg, &nc);
        else if (P->objective == ORC_OBJ_GATE_PAPER) {
            const int32_t front_ok = trk->prev_front ? trk->prev_front[(size_t)b * (P->N + 1) + t + 1] : 1;
            J += orc_gate_paper_step(P, trk, x, xn, xn + 10, &aux, gate0, front_ok, &marg, &nc);
        } else if (P->objective == ORC_OBJ_CONTOUR)
            J += orc_contour_step(P, trk, pa->s, pa->tan, pa->L, xn, xn + 10, &aux, &theta_prev);
        memcpy(x, xn, sizeof(double) * xdim);
    }
    if (P->objective == ORC_OBJ_TRACK)
        J += orc_track_state_term(P, x, trk->ref + 13 * (start + P->N));   /* eq.(8) terminal */

    if (margin) *margin = marg;
    if (ncross) *ncross = nc;
    if (aux_end) *aux_end = aux;
    if (x_end) memcpy(x_end, x, sizeof(double) * xdim);
    return J;
}

/* ------------------------------------------------------------------------------------------
 * Softmax weights eq.(4) PAPER.md:86-89 and weighted update eq.(5) PAPER.md:91-95.
 * The minimum is subtracted before the exponential (identical value, avoids overflow).
 * U^m = U* + dU^m (eq.(3)) and sum w = 1, so U*_new = u_nom + sum_k w_k du_k.
 * du is [K][N][4].
 * ---------------------------------------------------------------------------------------- */
void orc_weights_update(int32_t K, int32_t N, double lambda, const double* cost,
                        const double* du, const double* u_nom, double* weights, double* u_new)
{
    double beta = INFINITY;
    for (int k = 0; k < K; ++k) if (cost[k] < beta) beta = cost[k];
    double Z = 0.0;
    for (int k = 0; k < K; ++k) { weights[k] = exp(-(cost[k] - beta) / lambda); Z += weights[k]; }
    for (int k = 0; k < K; ++k) weights[k] /= Z;
    for (int j = 0; j < 4 * N; ++j) {
        double acc = 0.0;
        for (int k = 0; k < K; ++k) acc += weights[k] * du[(size_t)k * 4 * N + j];
        u_new[j] = u_nom[j] + acc;
    }
}

/* ------------------------------------------------------------------------------------------
 * One full MPPI iteration for B independent controllers (Alg. 1 lines 3-17).
 * Optional outputs (may be NULL): du_out [B][K][N][4], margin [B][K], ncross [B][K],
 * aux_end [B][K].  Returns 0, or -1 on a bad argument / allocation failure.
 * ---------------------------------------------------------------------------------------- */
int orc_step(const orc_params* P, const orc_track* trk, const double* x0 /*[B][13]*/,
             const int32_t* start /*[B]*/, const double* u_nom /*[B][N][4]*/, uint64_t seed,
             uint32_t iter, double* u_new /*[B][N][4]*/, double* cost /*[B][K]*/,
             double* weights /*[B][K]*/, double* du_out, double* margin, int32_t* ncross,
             int32_t* aux_end)
{
    if (!P || !trk || !x0 || !start || !u_nom || !u_new || !cost || !weights) return -1;
    const int K = P->K, N = P->N, B = P->B;
    orc_path_aux pa = { NULL, NULL, 0.0 };
    double* s = NULL; double* tan = NULL;
    if (P->objective == ORC_OBJ_CONTOUR_PAPER && (P->input_model != 1 || !trk->v_nom || !trk->v_new)) return -1;
    if (P->objective == ORC_OBJ_CONTOUR || P->objective == ORC_OBJ_CONTOUR_PAPER) {
        s = (double*)malloc(sizeof(double) * trk->P);
        tan = (double*)malloc(sizeof(double) * 3 * trk->P);
        if (!s || !tan) { free(s); free(tan); return -1; }
        pa.L = orc_path_prepare(trk->pts, trk->P, trk->closed, s, tan);
        pa.s = s; pa.tan = tan;
    }
    double* du_local = NULL;
    if (!du_out) {
        du_local = (double*)malloc(sizeof(double) * (size_t)K * N * 4);
        if (!du_local) { free(s); free(tan); return -1; }
    }
    orc_track trk5 = *trk;                       /* the fifth column needs its perturbations for eq.(5) */
    double* dv_local = NULL;
    if (P->objective == ORC_OBJ_CONTOUR_PAPER && !trk->dv_out) {
        dv_local = (double*)malloc(sizeof(double) * (size_t)B * K * N);
        if (!dv_local) { free(du_local); free(s); free(tan); return -1; }
        trk5.dv_out = dv_local;
    }
    trk = &trk5;
    for (int b = 0; b < B; ++b) {
        double* du = du_out ? du_out + (size_t)b * K * N * 4 : du_local;
        const double* un = u_nom + (size_t)b * N * 4;
#pragma omp parallel for schedule(static)
        for (int k = 0; k < K; ++k) {
            double mg; int32_t nc, ae;
            cost[(size_t)b * K + k] =
                orc_rollout_cost(P, trk, &pa, x0 + (P->objective == ORC_OBJ_CONTOUR_PAPER ? 19 : P->input_model == 1 ? 17 : 13) * b, start[b], un, seed, iter, (uint32_t)k,
                                 (uint32_t)b, du + (size_t)k * N * 4, &mg, &nc, &ae, NULL);
            /* [R-41] a rollout whose cost is not representable in the fp32 interface (NaN, or beyond 3.0e38: a
             * diverged sample) counts as cost 3.0e38 -- weight 0 unless every sample diverged (include/mppi.h) */
            if (!(fabs(cost[(size_t)b * K + k]) <= 3.0e38)) cost[(size_t)b * K + k] = 3.0e38;
            if (margin) margin[(size_t)b * K + k] = mg;
            if (ncross) ncross[(size_t)b * K + k] = nc;
            if (aux_end) aux_end[(size_t)b * K + k] = ae;
        }
        orc_weights_update(K, N, P->lambda, cost + (size_t)b * K, du, un,
                           weights + (size_t)b * K, u_new + (size_t)b * N * 4);
        if (P->objective == ORC_OBJ_CONTOUR_PAPER)            /* eq.(5) for the fifth input */
            for (int t = 0; t < N; ++t) {
                double acc = 0.0;
                for (int k = 0; k < K; ++k)
                    acc += weights[(size_t)b * K + k] * trk->dv_out[((size_t)b * K + k) * N + t];
                trk->v_new[(size_t)b * N + t] = trk->v_nom[(size_t)b * N + t] + acc;
            }
    }
    free(du_local); free(dv_local); free(s); free(tan);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Closed-loop glue of BASELINE.json configs[4] (receding horizon; Alg. 1
 * lines 2-3): apply u*_0 to the plant (the same RK4 model), advance the caller-owned start
 * index, shift the nominal by one step and repeat its last element [R-14].
 *   gate:    the plant segment is tested against the current gate exactly as in orc_gate_step;
 *            a valid pass advances start (mod G), a miss does not.
 *   track:   start <- min(start + 1, M - 1 - N)   (the reference clock advances one row)
 *   contour: start <- windowed nearest vertex to the new position (global if start was -1)
 * x [B][13] and start [B] are updated in place; u_nom_next [B][N][4] is written.
 * ---------------------------------------------------------------------------------------- */
int orc_sim_step(const orc_params* P, const orc_track* trk, double* x, int32_t* start,
                 const double* u_new, double* u_nom_next)
{
    if (!P || !trk || !x || !start || !u_new || !u_nom_next) return -1;
    const int N = P->N;
    for (int b = 0; b < P->B; ++b) {
        const int rate = P->input_model == 1, xdim = rate ? 17 : 13;   /* [R-27]: rows of 17 */
        double* xb = x + xdim * b;
        const double* ub = u_new + (size_t)b * N * 4;
        double xn[17];
        if (rate) orc_rk4_rate_step(P, xb, ub, P->dt, xn);
        else orc_rk4_step(P, xb, ub, P->dt, xn);
        if (P->objective == ORC_OBJ_GATE || P->objective == ORC_OBJ_GATE_PAPER) {
            int32_t gate = start[b];
            (void)orc_gate_step(P, trk, xb, xn, xn + 10, &gate, NULL, NULL);
            start[b] = gate;
        } else if (P->objective == ORC_OBJ_TRACK) {
            int32_t nxt = start[b] + 1;
            if (nxt > trk->M - 1 - N) nxt = trk->M - 1 - N;
            start[b] = nxt;
        } else {
            start[b] = orc_path_nearest(trk->pts, trk->P, trk->closed, xn, start[b], P->window);
        }
        memcpy(xb, xn, sizeof(double) * xdim);
        double* nn = u_nom_next + (size_t)b * N * 4;
        for (int t = 0; t < N; ++t) {
            const int src = (t + 1 < N) ? t + 1 : N - 1;
            for (int i = 0; i < 4; ++i) nn[4 * t + i] = ub[4 * src + i];
        }
    }
    return 0;
}

/* Closed-loop glue under ORC_OBJ_CONTOUR_PAPER [R-39]: rows of 19.  The drone part of the state takes one
 * rate-model RK4 step with u_new[b][0] (as orc_sim_step); the progress states are the controller's own
 * (virtual) states and advance by [R-34] with the optimised v_new[b][0]; both nominals shift by one step
 * with the last entry repeated [R-14].  start is not used by this objective (the path is looked up by
 * theta) and is left alone.  x [B][19] is updated in place. */
int orc_sim_step_progress(const orc_params* P, double* x, const double* u_new, double* u_nom_next,
                          const double* v_new, double* v_nom_next)
{
    if (!P || !x || !u_new || !u_nom_next || !v_new || !v_nom_next) return -1;
    if (P->objective != ORC_OBJ_CONTOUR_PAPER || P->input_model != 1) return -2;
    const int N = P->N;
    for (int b = 0; b < P->B; ++b) {
        double* xb = x + 19 * b;
        const double* ub = u_new + (size_t)b * N * 4;
        const double* vb = v_new + (size_t)b * N;
        double xn[19];
        orc_rk4_rate_step(P, xb, ub, P->dt, xn);
        orc_progress_step(P, xb[17], xb[18], vb[0], &xn[17], &xn[18]);
        memcpy(xb, xn, sizeof(xn));
        for (int t = 0; t < N; ++t) {
            const int src = (t + 1 < N) ? t + 1 : N - 1;
            for (int i = 0; i < 4; ++i) u_nom_next[((size_t)b * N + t) * 4 + i] = ub[4 * src + i];
        }
        for (int t = 0; t < N; ++t) v_nom_next[(size_t)b * N + t] = vb[(t + 1 < N) ? t + 1 : N - 1];
    }
    return 0;
}

/* Threads the sample loop will use (reported by bench.py's cpu_baseline). */
int orc_num_threads(void)
{
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp single
        n = omp_get_num_threads();
    }
#endif
    return n;
}
