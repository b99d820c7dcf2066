// mppi_cost.cuh -- the three per-step objectives (section IV) as register-resident
// accumulators.  Track data (gates / reference rows / path) is read from shared memory.
#pragma once
#include "mppi_device.cuh"

namespace mppi {

enum { OBJ_GATE = 0, OBJ_TRACK = 1, OBJ_CONTOUR = 2, OBJ_GATE_PAPER = 3, OBJ_CONTOUR_PAPER = 4 };

// ---- gate progress: eq.(6) PAPER.md:105-110 with un-squared distances [D-2], in-horizon target
// switching PAPER.md:112, geometric pass test [R-9],[R-10]; constants BASELINE.json configs[0].
//
// The progress sum telescopes while the target does not change: sum_t (d_t - d_{t-1}) = d_end -
// d_begin of each constant-target segment.  Only the signed plane distance s = n.(p - c) is needed
// every step (the crossing test); the distances are taken at a target switch and at the horizon end.
// s is evaluated as n.p - (n.c) with the plane offset n.c formed in double by mppi_set_gates (three
// FFMAs per step instead of three subtractions and three multiply-adds; the rounding of the
// cancellation, <= ~1e-6 m at |c| ~ 13 m, is of the size of the fp32 position error itself and a
// tenth of the 1e-5 m crossing margin of north_star).
// The body-rate term accumulates sum |omega|^2 and is scaled once at the end.
struct GateCost {
    int gate;                 // current target
    float d0;                 // |p - c| where the current segment began
    float s_prev;             // n . (p_{t-1} - c)
    float ppx, ppy, ppz;      // p_{t-1}
    float J;                  // pass bonuses / miss penalties / finished segments
    float w2;                 // sum_t |omega_t|^2

    template <int MATH>
    __device__ __forceinline__ static float norm3(float x, float y, float z)
    {
        const float r2 = fmaf(z, z, fmaf(y, y, x * x));
        return MATH == 0 ? sqrtf(r2) : mufu_sqrt(r2);
    }
    __device__ __forceinline__ static float plane(const float4 n, const float nc, float px, float py, float pz)
    {
        return fmaf(n.z, pz, fmaf(n.y, py, fmaf(n.x, px, -nc)));
    }
    template <int MATH>
    __device__ __forceinline__ void retarget(const float4* s_gates, float px, float py, float pz)
    {
        const float4 c = s_gates[4 * gate], n = s_gates[4 * gate + 1];
        d0 = norm3<MATH>(px - c.x, py - c.y, pz - c.z);
        s_prev = plane(n, s_gates[4 * gate + 2].w, px, py, pz);
    }
    template <int MATH>
    __device__ __forceinline__ void init(const DevParams& P, const float4* s_gates, int start, const State& x)
    {
        gate = wrap_index(start, P.G);
        J = 0.0f; w2 = 0.0f;
        ppx = x.px; ppy = x.py; ppz = x.pz;
        retarget<MATH>(s_gates, x.px, x.py, x.pz);
    }
    // post-step state x_{t+1}
    template <int MATH>
    __device__ __forceinline__ void step(const DevParams& P, const float4* s_gates, const State& x)
    {
        const float4 n = s_gates[4 * gate + 1], h = s_gates[4 * gate + 2];
        const float s = plane(n, h.w, x.px, x.py, x.pz);
        if (s_prev < 0.0f && s >= 0.0f) {                 // front -> back through the plane
            const float4 c = s_gates[4 * gate], v = s_gates[4 * gate + 3];
            const float ax = x.px - c.x, ay = x.py - c.y, az = x.pz - c.z;
            const float alpha = s_prev / (s_prev - s);
            const float rx = ppx - c.x, ry = ppy - c.y, rz = ppz - c.z;
            const float hx = fmaf(alpha, ax - rx, rx), hy = fmaf(alpha, ay - ry, ry), hz = fmaf(alpha, az - rz, rz);
            const float y = fmaf(h.z, hz, fmaf(h.y, hy, h.x * hx));
            const float z = fmaf(v.z, hz, fmaf(v.y, hy, v.x * hx));
            if (fabsf(y) <= c.w && fabsf(z) <= n.w) {     // inside the opening: pass + switch
                J += (norm3<MATH>(ax, ay, az) - d0) - P.bonus;        // close the segment
                gate = (gate + 1 == P.G) ? 0 : gate + 1;
                retarget<MATH>(s_gates, x.px, x.py, x.pz);            // new target from the next step on
            } else {                                      // miss: target unchanged
                J += P.miss;
                s_prev = s;
            }
        } else {
            s_prev = s;
        }
        ppx = x.px; ppy = x.py; ppz = x.pz;
        w2 = fmaf(x.oz, x.oz, fmaf(x.oy, x.oy, fmaf(x.ox, x.ox, w2)));
    }
    template <int MATH>
    __device__ __forceinline__ float finish(const DevParams& P, const float4* s_gates, const State& x) const
    {
        const float4 c = s_gates[4 * gate];
        const float d = norm3<MATH>(x.px - c.x, x.py - c.y, x.pz - c.z);
        return fmaf(P.w_omega, w2, J + (d - d0));
    }
};

// ---- the paper's own gate progress: eq.(6),(7) PAPER.md:105-129 with SQUARED distances [R-23], the
// conditional near-gate term Q_near |p_k - c|^2 for |p_k - c| < r_near on the pre-step state [R-24],
// and the temporal gate-switching check of Fig. 2 [R-25]: a geometric pass of the
// horizon's START gate at state index t+1 registers only if the caller's previous-iteration flag
// front[t+1] is set; later gates of the horizon switch on geometry alone.  As in GateCost the
// progress sum telescopes per constant-target segment (here without any square root).
// s_front: N+1 ints in shared memory (all ones when the caller gave no flags).
struct GatePaperCost {
    int gate, gate0;
    float d2_0;               // |p - c|^2 where the current segment began
    float d2_prev;            // |p_t - c|^2 of the pre-step state against the current target
    float s_prev;             // n . (p_t - c)
    float ppx, ppy, ppz;      // p_t
    float J;                  // bonuses / penalties / near terms / finished segments
    float w2;                 // sum_t |omega_t|^2

    __device__ __forceinline__ void retarget(const float4* s_gates, float px, float py, float pz)
    {
        const float4 c = s_gates[4 * gate], n = s_gates[4 * gate + 1];
        const float rx = px - c.x, ry = py - c.y, rz = pz - c.z;
        d2_0 = fmaf(rz, rz, fmaf(ry, ry, rx * rx));
        d2_prev = d2_0;
        s_prev = fmaf(n.z, rz, fmaf(n.y, ry, n.x * rx));
    }
    __device__ __forceinline__ void init(const DevParams& P, const float4* s_gates, int start, const State& x)
    {
        gate = wrap_index(start, P.G);
        gate0 = gate;
        J = 0.0f; w2 = 0.0f;
        ppx = x.px; ppy = x.py; ppz = x.pz;
        retarget(s_gates, x.px, x.py, x.pz);
    }
    // post-step state x_{t+1} of step t
    __device__ __forceinline__ void step(const DevParams& P, const float4* s_gates, const int* s_front,
                                         const State& x, int t)
    {
        // eq.(7) on the pre-step state p_t: against the step's own target [R-24], or (near_mode 1, [R-40]) against
        // the horizon's start gate also once the target has moved on
        float dn2 = d2_prev;
        if (P.near_mode == 1 && gate != gate0) {
            const float4 c0 = s_gates[4 * gate0];
            const float ux = ppx - c0.x, uy = ppy - c0.y, uz = ppz - c0.z;
            dn2 = fmaf(uz, uz, fmaf(uy, uy, ux * ux));
        }
        if (dn2 < P.r_near2) J = fmaf(P.q_near, dn2, J);
        const float4 c = s_gates[4 * gate], n = s_gates[4 * gate + 1];
        const float ax = x.px - c.x, ay = x.py - c.y, az = x.pz - c.z;
        const float d2 = fmaf(az, az, fmaf(ay, ay, ax * ax));
        const float s = fmaf(n.z, az, fmaf(n.y, ay, n.x * ax));
        bool switched = false;
        if (s_prev < 0.0f && s >= 0.0f) {                 // front -> back through the plane
            const float4 h = s_gates[4 * gate + 2], v = s_gates[4 * gate + 3];
            const float alpha = s_prev / (s_prev - s);
            const float rx = ppx - c.x, ry = ppy - c.y, rz = ppz - c.z;
            const float hx = fmaf(alpha, ax - rx, rx), hy = fmaf(alpha, ay - ry, ry), hz = fmaf(alpha, az - rz, rz);
            const float y = fmaf(h.z, hz, fmaf(h.y, hy, h.x * hx));
            const float z = fmaf(v.z, hz, fmaf(v.y, hy, v.x * hx));
            if (fabsf(y) <= c.w && fabsf(z) <= n.w) {
                if (gate != gate0 || s_front[t + 1] != 0) {           // temporally consistent pass
                    J += (d2 - d2_0) - P.bonus;                       // close the segment
                    gate = (gate + 1 == P.G) ? 0 : gate + 1;
                    retarget(s_gates, x.px, x.py, x.pz);              // new target from the next step on
                    switched = true;
                }
            } else {
                J += P.miss;                                          // miss: target unchanged
            }
        }
        if (!switched) { s_prev = s; d2_prev = d2; }
        ppx = x.px; ppy = x.py; ppz = x.pz;
        w2 = fmaf(x.oz, x.oz, fmaf(x.oy, x.oy, fmaf(x.ox, x.ox, w2)));
    }
    __device__ __forceinline__ float finish(const DevParams& P) const
    {
        return fmaf(P.w_omega, w2, J + (d2_prev - d2_0));
    }
};

// ---- trajectory tracking: eq.(8), [R-11] ------------------------------------
// s_ref holds rows t0 .. t0+N of the reference, 4 float4 per row.
__device__ __forceinline__ float track_state_term(const DevParams& P, const float4* row, const State& x)
{
    const float4 a = row[0], b = row[1], c = row[2], d = row[3];
    // a = (p, qw)  b = (qx qy qz, vx)  c = (vy vz, wx wy)  d = (wz, -, -, -)
    const float ex = x.px - a.x, ey = x.py - a.y, ez = x.pz - a.z;
    const float dot = x.qw * a.w + x.qx * b.x + x.qy * b.y + x.qz * b.z;
    const float sg = dot < 0.0f ? -1.0f : 1.0f;           // double cover: compare with +-q_ref
    const float q0 = fmaf(-sg, a.w, x.qw), q1 = fmaf(-sg, b.x, x.qx), q2 = fmaf(-sg, b.y, x.qy),
                q3 = fmaf(-sg, b.z, x.qz);
    const float ux = x.vx - b.w, uy = x.vy - c.x, uz = x.vz - c.y;
    const float wx = x.ox - c.z, wy = x.oy - c.w, wz = x.oz - d.x;
    float J = P.Qp * (ex * ex + ey * ey + ez * ez);
    J = fmaf(P.Qv, ux * ux + uy * uy + uz * uz, J);
    J = fmaf(P.Qq, q0 * q0 + q1 * q1 + q2 * q2 + q3 * q3, J);
    J = fmaf(P.Qw, wx * wx + wy * wy + wz * wz, J);
    return J;
}

__device__ __forceinline__ float track_stage(const DevParams& P, const float4* row, const State& x,
                                             const float4 T)
{
    const float a = T.x - P.hover, b = T.y - P.hover, c = T.z - P.hover, d = T.w - P.hover;
    return fmaf(P.R, a * a + b * b + c * c + d * d, track_state_term(P, row, x));
}

// ---- contouring: eq.(9) PAPER.md:149-161 in the projection variant of configs[3] [D-6] ---------
// s_path holds all P points (P_i, s_i), then all P tangents (t_i, 0).
struct ContourCost {
    int idx;
    float theta_prev;

    // nearest vertex among offsets -W..+W around `centre`, first minimiser in scan order [R-12]
    __device__ __forceinline__ static int nearest(const DevParams& P, const float4* s_path,
                                                  int centre, float px, float py, float pz)
    {
        float best = __int_as_float(0x7f800000);
        int ibest = centre;
        if (P.closed) {
            int i = wrap_index(centre - P.window, P.P);
            for (int o = -P.window; o <= P.window; ++o) {
                const float4 q = s_path[i];
                const float dx = px - q.x, dy = py - q.y, dz = pz - q.z;
                const float d2 = dx * dx + dy * dy + dz * dz;
                if (d2 < best) { best = d2; ibest = i; }
                i = (i + 1 == P.P) ? 0 : i + 1;
            }
        } else {
            const int lo = max(centre - P.window, 0), hi = min(centre + P.window, P.P - 1);
            for (int i = lo; i <= hi; ++i) {
                const float4 q = s_path[i];
                const float dx = px - q.x, dy = py - q.y, dz = pz - q.z;
                const float d2 = dx * dx + dy * dy + dz * dz;
                if (d2 < best) { best = d2; ibest = i; }
            }
        }
        return ibest;
    }
    // The same search on the padded copy of the points that stage_inputs<OBJ_CONTOUR> appends to the path in
    // shared memory: ext[j] = point (j - W), wrapped on a closed path, a far sentinel (distance inf, never
    // the minimum) beyond the ends of an open one, ext = s_path + 2 P.  The window of `centre` is then the
    // contiguous run ext[centre .. centre + 2W]: no wrap test per candidate, and with the window known at
    // compile time (WFIX = 16, the default) every load has an immediate offset and is independent of the
    // others.  Four runs of the window are scanned independently and merged in scan order -- a later
    // run wins only when strictly smaller -- which keeps [R-12]'s first minimiser with a four times
    // shorter dependency chain.  Distances are formed exactly as in nearest().
    static constexpr int kExtPad = 7;     // extra entries before and after the padded copy (nearest_rot)
    template <int LO, int HI>
    __device__ __forceinline__ static void scan_run(const float4* w, float px, float py, float pz, float& best, int& ob)
    {
#pragma unroll
        for (int o = LO; o < HI; ++o) {
            const float4 q = w[o];
            const float dx = px - q.x, dy = py - q.y, dz = pz - q.z;
            const float d2 = dx * dx + dy * dy + dz * dz;
            if (d2 < best) { best = d2; ob = o; }
        }
    }
    template <int WFIX>
    __device__ __forceinline__ static int nearest_ext(const DevParams& P, const float4* s_path, int centre,
                                                      float px, float py, float pz)
    {
        const int W = WFIX > 0 ? WFIX : P.window;
        const float4* w = s_path + 2 * P.P + kExtPad + centre;
        const float inf = __int_as_float(0x7f800000);
        float best = inf;
        int ob = W;
        if (WFIX > 0) {
            constexpr int n = 2 * WFIX + 1, g = (n + 3) / 4;
            float b1 = inf, b2 = inf, b3 = inf;
            int o1 = g, o2 = 2 * g, o3 = 3 * g;
            scan_run<0, g>(w, px, py, pz, best, ob);
            scan_run<g, 2 * g>(w, px, py, pz, b1, o1);
            scan_run<2 * g, 3 * g>(w, px, py, pz, b2, o2);
            scan_run<3 * g, n>(w, px, py, pz, b3, o3);
            if (b1 < best) { best = b1; ob = o1; }
            if (b2 < best) { best = b2; ob = o2; }
            if (b3 < best) { best = b3; ob = o3; }
        } else {
            for (int o = 0; o <= 2 * W; ++o) {
                const float4 q = w[o];
                const float dx = px - q.x, dy = py - q.y, dz = pz - q.z;
                const float d2 = dx * dx + dy * dy + dz * dz;
                if (d2 < best) { best = d2; ob = o; }
            }
        }
        int i = centre + ob - W;
        if (P.closed) { if (i < 0) i += P.P; else if (i >= P.P) i -= P.P; }
        return i;
    }
    // Bank-conflict-free form for the throughput kernels (window 16): a 128-bit shared load is served per
    // quarter-warp, 8 lanes x 16 B over the 32 banks, and is conflict-free when the 8 vertex indices are
    // distinct mod 8.  Each lane therefore starts its scan at the last entry at or before its window whose
    // index is congruent to its lane number mod 8 (r <= 7 entries early) and walks 40 entries instead of
    // 33; entry o belongs to the window iff r <= o <= r + 32, which only the first and the last seven
    // need to test.  Scan order, strict comparison and distances are those of nearest(): same minimiser.
    __device__ __forceinline__ static int nearest_rot(const DevParams& P, const float4* s_path, int centre,
                                                      float px, float py, float pz)
    {
        constexpr int W = 16, n = 2 * W + 1;
        const int ws = centre + kExtPad;                         // window start in the padded copy
        const int r = (ws - (int)(threadIdx.x & 7)) & 7;
        const float4* w = s_path + 2 * P.P + (ws - r);
        const float inf = __int_as_float(0x7f800000);
        float best = inf;
        int ob = W + r;
#pragma unroll
        for (int o = 0; o < n + kExtPad; ++o) {
            const float4 q = w[o];
            const float dx = px - q.x, dy = py - q.y, dz = pz - q.z;
            float d2 = dx * dx + dy * dy + dz * dz;
            if (o < kExtPad) d2 = o >= r ? d2 : inf;
            if (o >= n) d2 = o <= r + 2 * W ? d2 : inf;
            if (d2 < best) { best = d2; ob = o; }
        }
        int i = centre + (ob - r) - W;
        if (P.closed) { if (i < 0) i += P.P; else if (i >= P.P) i -= P.P; }
        return i;
    }
    __device__ __forceinline__ static int nearest_smem(const DevParams& P, const float4* s_path, int centre,
                                                       float px, float py, float pz)
    {
        return P.window == 16 ? nearest_ext<16>(P, s_path, centre, px, py, pz) : nearest_ext<0>(P, s_path, centre, px, py, pz);
    }
    // lag error e_l, contour error squared e_c^2, progress theta = s_i + e_l
    __device__ __forceinline__ static void project(const DevParams& P, const float4* s_path, int i, float px, float py,
                                                   float pz, float& e_l, float& e_c2, float& theta)
    {
        const float4 q = s_path[i], t = s_path[P.P + i];
        const float dx = px - q.x, dy = py - q.y, dz = pz - q.z;
        e_l = dx * t.x + dy * t.y + dz * t.z;
        e_c2 = fmaxf((dx * dx + dy * dy + dz * dz) - e_l * e_l, 0.0f);
        theta = q.w + e_l;
    }
    // i0 is the block-wide initial index (global or windowed search done by the caller)
    __device__ __forceinline__ void init(const DevParams& P, const float4* s_path, int i0, const State& x)
    {
        float e_l, e_c2;
        idx = i0;
        project(P, s_path, i0, x.px, x.py, x.pz, e_l, e_c2, theta_prev);
    }
    template <bool ROT = false>
    __device__ __forceinline__ float step(const DevParams& P, const float4* s_path, const State& x)
    {
        return step_at<ROT>(P, s_path, x.px, x.py, x.pz, x.ox * x.ox + x.oy * x.oy + x.oz * x.oz);
    }
    // the same step from a position and |omega|^2 (what the rollout warps of the latency kernel hand over)
    template <bool ROT = false>
    __device__ __forceinline__ float step_at(const DevParams& P, const float4* s_path, const float px, const float py,
                                             const float pz, const float w2)
    {
        idx = (ROT && P.window == 16) ? nearest_rot(P, s_path, idx, px, py, pz)
                                      : nearest_smem(P, s_path, idx, px, py, pz);
        return step_found(P, s_path, px, py, pz, w2);
    }
    // the cost of the step once idx holds the nearest vertex of this position
    __device__ __forceinline__ float step_found(const DevParams& P, const float4* s_path, const float px, const float py,
                                                const float pz, const float w2)
    {
        float e_l, e_c2, theta;
        project(P, s_path, idx, px, py, pz, e_l, e_c2, theta);
        float d = theta - theta_prev;
        if (P.closed) d -= P.path_L * ceilf((d - 0.5f * P.path_L) * P.inv_path_L);  // (-L/2, L/2]
        theta_prev = theta;
        float J = P.q_c * e_c2;
        J = fmaf(P.q_l, e_l * e_l, J);
        J = fmaf(-P.mu, d, J);
        return fmaf(P.w_omega, w2, J);
    }
};

}  // namespace mppi
