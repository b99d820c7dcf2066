// mppi_cost.cuh -- the three per-step objectives (section IV) as register-resident
// accumulators.  Track data (gates / reference rows / path) is read from shared memory.
#pragma once
#include "mppi_device.cuh"

namespace mppi {

enum { OBJ_GATE = 0, OBJ_TRACK = 1, OBJ_CONTOUR = 2 };

// ---- gate progress: eq.(6) PAPER.md:105-110 with un-squared distances [D-2], in-horizon target
// switching PAPER.md:112, geometric pass test [R-9],[R-10]; constants BASELINE.json configs[0].
struct GateCost {
    int gate;                 // current target
    float rx, ry, rz;         // p_{t-1} - c
    float d_prev, s_prev;     // |p_{t-1} - c|, n . (p_{t-1} - c)

    __device__ __forceinline__ void retarget(const float4* s_gates, float px, float py, float pz)
    {
        const float4 c = s_gates[4 * gate], n = s_gates[4 * gate + 1];
        rx = px - c.x; ry = py - c.y; rz = pz - c.z;
        d_prev = sqrtf(rx * rx + ry * ry + rz * rz);
        s_prev = n.x * rx + n.y * ry + n.z * rz;
    }
    __device__ __forceinline__ void init(const DevParams& P, const float4* s_gates, int start,
                                         const State& x)
    {
        gate = wrap_index(start, P.G);
        retarget(s_gates, x.px, x.py, x.pz);
    }
    // post-step state x_{t+1}; returns the step cost
    __device__ __forceinline__ float step(const DevParams& P, const float4* s_gates, const State& x)
    {
        const float4 c = s_gates[4 * gate], n = s_gates[4 * gate + 1];
        const float ax = x.px - c.x, ay = x.py - c.y, az = x.pz - c.z;
        const float d = sqrtf(ax * ax + ay * ay + az * az);
        const float s = n.x * ax + n.y * ay + n.z * az;
        float J = d - d_prev;
        if (s_prev < 0.0f && s >= 0.0f) {                 // front -> back through the plane
            const float4 h = s_gates[4 * gate + 2], v = s_gates[4 * gate + 3];
            const float alpha = s_prev / (s_prev - s);
            const float hx = fmaf(alpha, ax - rx, rx), hy = fmaf(alpha, ay - ry, ry),
                        hz = fmaf(alpha, az - rz, rz);
            const float y = h.x * hx + h.y * hy + h.z * hz;
            const float z = v.x * hx + v.y * hy + v.z * hz;
            if (fabsf(y) <= c.w && fabsf(z) <= n.w) {     // inside the opening: pass + switch
                J -= P.bonus;
                gate = (gate + 1 == P.G) ? 0 : gate + 1;
                retarget(s_gates, x.px, x.py, x.pz);      // the new target applies from the next step
            } else {                                      // miss: target unchanged
                J += P.miss;
                rx = ax; ry = ay; rz = az; d_prev = d; s_prev = s;
            }
        } else {
            rx = ax; ry = ay; rz = az; d_prev = d; s_prev = s;
        }
        return fmaf(P.w_omega, x.ox * x.ox + x.oy * x.oy + x.oz * x.oz, J);
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
// s_path holds all P points: (P_i, s_i), (t_i, 0).
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
                const float4 q = s_path[2 * i];
                const float dx = px - q.x, dy = py - q.y, dz = pz - q.z;
                const float d2 = dx * dx + dy * dy + dz * dz;
                if (d2 < best) { best = d2; ibest = i; }
                i = (i + 1 == P.P) ? 0 : i + 1;
            }
        } else {
            const int lo = max(centre - P.window, 0), hi = min(centre + P.window, P.P - 1);
            for (int i = lo; i <= hi; ++i) {
                const float4 q = s_path[2 * i];
                const float dx = px - q.x, dy = py - q.y, dz = pz - q.z;
                const float d2 = dx * dx + dy * dy + dz * dz;
                if (d2 < best) { best = d2; ibest = i; }
            }
        }
        return ibest;
    }
    // lag error e_l, contour error squared e_c^2, progress theta = s_i + e_l
    __device__ __forceinline__ static void project(const float4* s_path, int i, float px, float py,
                                                   float pz, float& e_l, float& e_c2, float& theta)
    {
        const float4 q = s_path[2 * i], t = s_path[2 * i + 1];
        const float dx = px - q.x, dy = py - q.y, dz = pz - q.z;
        e_l = dx * t.x + dy * t.y + dz * t.z;
        e_c2 = fmaxf((dx * dx + dy * dy + dz * dz) - e_l * e_l, 0.0f);
        theta = q.w + e_l;
    }
    // i0 is the block-wide initial index (global or windowed search done by the caller)
    __device__ __forceinline__ void init(const float4* s_path, int i0, const State& x)
    {
        float e_l, e_c2;
        idx = i0;
        project(s_path, i0, x.px, x.py, x.pz, e_l, e_c2, theta_prev);
    }
    __device__ __forceinline__ float step(const DevParams& P, const float4* s_path, const State& x)
    {
        idx = nearest(P, s_path, idx, x.px, x.py, x.pz);
        float e_l, e_c2, theta;
        project(s_path, idx, x.px, x.py, x.pz, e_l, e_c2, theta);
        float d = theta - theta_prev;
        if (P.closed) d -= P.path_L * ceilf((d - 0.5f * P.path_L) * P.inv_path_L);  // (-L/2, L/2]
        theta_prev = theta;
        float J = P.q_c * e_c2;
        J = fmaf(P.q_l, e_l * e_l, J);
        J = fmaf(-P.mu, d, J);
        return fmaf(P.w_omega, x.ox * x.ox + x.oy * x.oy + x.oz * x.oz, J);
    }
};

}  // namespace mppi
