"""Seeded synthetic inputs for the five BASELINE.json configs (plus stress cases).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the
method's arithmetic: no Philox, no dynamics, no cost, no softmax.  It only builds tracks,
references, paths, initial states and parameter sets from the recipes in DESIGN.md section
"Input recipe" (readings R-15/R-16).  It stands in for the paper's Circle /
Figure-8 / Split-S tracks and CPC references, whose coordinates are not
printed in the paper.

Every array is rounded to float32 so that the GPU (fp32) and the oracle (fp64) see the same
real numbers; scalars in `params` are float32-representable for the same reason.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

OBJ_GATE, OBJ_TRACK, OBJ_CONTOUR, OBJ_GATE_PAPER, OBJ_CONTOUR_PAPER = 0, 1, 2, 3, 4


def _f32(v):
    return float(np.float32(v))


def base_params(**over) -> dict:
    """Quadrotor + cost constants of BASELINE.json configs[0]/[2]/[3]; all float32-exact."""
    p = dict(K=256, N=20, B=1, objective=OBJ_GATE,
             dt=0.02, sigma=1.0, mass=0.85, Jx=1e-3, Jy=1e-3, Jz=1.7e-3, arm=0.15, c_tau=0.016,
             g=9.81, T_min=0.0, T_max=7.0, w_omega=0.01, gate_miss_penalty=10.0,
             gate_pass_bonus=5.0, Qp=100.0, Qv=1.0, Qq=10.0, Qw=0.1, R=0.01, q_contour=200.0,
             q_lag=50.0, mu_progress=2.0, window=16, q_near=0.0, r_near=0.0,
             input_model=0, rate_max=0.0, drag_x=0.0, drag_y=0.0, drag_z=0.0, w_limit=0.0, omega_max=0.0,
             sigma_v=0.0, dv_max=0.0, v_theta_max=0.0, r_dv=0.0, near_mode=0)
    p["lambda"] = 1.0
    p.update(over)
    for k, v in p.items():
        if k not in ("K", "N", "B", "objective", "window", "input_model", "near_mode"):
            p[k] = _f32(v)
    return p


def hover_thrust(p: dict) -> np.float32:
    """Nominal input of the configs: each rotor carries a quarter of the weight."""
    return np.float32(np.float32(p["mass"]) * np.float32(p["g"]) / np.float32(4.0))


@dataclass
class Workload:
    name: str
    params: dict
    x0: np.ndarray                      # [B,13] f32: p, q(wxyz), v, omega
    start: np.ndarray                   # [B] i32
    u_nom: np.ndarray                   # [B,N,4] f32
    gates: np.ndarray | None = None     # [G,11] f32
    ref: np.ndarray | None = None       # [M,13] f32
    path: np.ndarray | None = None      # [P,3] f32
    prev_front: np.ndarray | None = None  # [B,N+1] i32, objective 3 only (None = all in front)
    v_nom: np.ndarray | None = None     # [B,N] f32, objective 4 only: nominal progress accelerations
    closed: bool = True
    seed: int = 0
    iters: int = 1                      # optimiser iterations (cfg1) or control steps (cfg4)
    notes: dict = field(default_factory=dict)


# ---- tracks ------------------------------------------------------------------------------

def _gate_rows(centres, normals, half_w, half_h):
    n = np.asarray(normals, dtype=np.float64)
    n = n / np.linalg.norm(n, axis=1, keepdims=True)
    h = np.stack([n[:, 1], -n[:, 0], np.zeros(len(n))], axis=1)   # h = (n_y, -n_x, 0): h x n = +z
    h = h / np.linalg.norm(h, axis=1, keepdims=True)
    g = np.concatenate([np.asarray(centres, dtype=np.float64), n, h,
                        np.full((len(n), 1), half_w), np.full((len(n), 1), half_h)], axis=1)
    return g.astype(np.float32)


def circle_gates(n_gates=4, radius=5.0, z=1.5, width=1.5):
    """configs[0]: square gates on a circle, normals tangent (counter-clockwise travel)."""
    a = 2.0 * np.pi * np.arange(n_gates) / n_gates
    c = np.stack([radius * np.cos(a), radius * np.sin(a), np.full(n_gates, z)], axis=1)
    n = np.stack([-np.sin(a), np.cos(a), np.zeros(n_gates)], axis=1)
    return _gate_rows(c, n, width / 2, width / 2)


def lemniscate_gates(n_gates=7, a=12.0, width=1.5, height_seed=1):
    """configs[1]: gates on a Bernoulli lemniscate at t_i = 2 pi i / n, normal = unit tangent,
    heights uniform in [1,3] m from numpy default_rng(height_seed)  [R-16]."""
    t = 2.0 * np.pi * np.arange(n_gates) / n_gates
    den = 1.0 + np.sin(t) ** 2
    x = a * np.cos(t) / den
    y = a * np.sin(t) * np.cos(t) / den
    dden = 2.0 * np.sin(t) * np.cos(t)
    dx = a * (-np.sin(t) * den - np.cos(t) * dden) / den ** 2
    dy = a * ((np.cos(t) ** 2 - np.sin(t) ** 2) * den - np.sin(t) * np.cos(t) * dden) / den ** 2
    z = np.random.default_rng(height_seed).uniform(1.0, 3.0, n_gates)
    c = np.stack([x, y, z], axis=1)
    n = np.stack([dx, dy, np.zeros(n_gates)], axis=1)
    return _gate_rows(c, n, width / 2, width / 2)


def lissajous_reference(n_rows, dt, g=9.81):
    """configs[2]: p(t) = (10 sin .6t, 6 sin 1.2t, 2 + .5 sin .3t); v, a, jerk in closed form;
    attitude from differential flatness with yaw 0; body rates from the jerk (yaw rate 0)."""
    t = np.arange(n_rows) * float(dt)
    A = np.array([10.0, 6.0, 0.5]); W = np.array([0.6, 1.2, 0.3]); off = np.array([0.0, 0.0, 2.0])
    p = A * np.sin(np.outer(t, W)) + off
    v = A * W * np.cos(np.outer(t, W))
    acc = -A * W ** 2 * np.sin(np.outer(t, W))
    jerk = -A * W ** 3 * np.cos(np.outer(t, W))
    rows = np.zeros((n_rows, 13))
    for i in range(n_rows):
        f = acc[i] + np.array([0.0, 0.0, g])
        fn = np.linalg.norm(f)
        zb = f / fn
        xc = np.array([1.0, 0.0, 0.0])
        yb = np.cross(zb, xc); yb /= np.linalg.norm(yb)
        xb = np.cross(yb, zb)
        Rm = np.stack([xb, yb, zb], axis=1)
        q = _rot_to_quat(Rm)
        hw = (jerk[i] - np.dot(zb, jerk[i]) * zb) / fn
        om = np.array([-np.dot(hw, yb), np.dot(hw, xb), 0.0])
        rows[i] = np.concatenate([p[i], q, v[i], om])
    return rows.astype(np.float32)


def _rot_to_quat(R):
    tr = np.trace(R)
    if tr > 0:
        s = np.sqrt(tr + 1.0) * 2
        q = np.array([0.25 * s, (R[2, 1] - R[1, 2]) / s, (R[0, 2] - R[2, 0]) / s,
                      (R[1, 0] - R[0, 1]) / s])
    else:
        i = int(np.argmax(np.diag(R)))
        j, k = (i + 1) % 3, (i + 2) % 3
        s = np.sqrt(1.0 + R[i, i] - R[j, j] - R[k, k]) * 2
        q = np.zeros(4)
        q[0] = (R[k, j] - R[j, k]) / s
        q[1 + i] = 0.25 * s
        q[1 + j] = (R[j, i] + R[i, j]) / s
        q[1 + k] = (R[k, i] + R[i, k]) / s
    q = q / np.linalg.norm(q)
    return q if q[0] >= 0 else -q


def spline_path(centres, n_points=500, dense=20001):
    """configs[3]: periodic cubic spline through the gate centres, resampled to n_points
    uniformly spaced in arc length (the end point is not repeated)  [R-13]."""
    from scipy.interpolate import CubicSpline
    c = np.asarray(centres, dtype=np.float64)
    pts = np.concatenate([c, c[:1]], axis=0)
    chord = np.concatenate([[0.0], np.cumsum(np.linalg.norm(np.diff(pts, axis=0), axis=1))])
    cs = CubicSpline(chord, pts, bc_type="periodic")
    u = np.linspace(0.0, chord[-1], dense)
    d = cs(u)
    s = np.concatenate([[0.0], np.cumsum(np.linalg.norm(np.diff(d, axis=0), axis=1))])
    target = np.arange(n_points) * (s[-1] / n_points)
    uu = np.interp(target, s, u)
    return cs(uu).astype(np.float32)


# ---- the five configs ----------------------------------------------------------------------

def _level_state(p, v=(0, 0, 0)):
    x = np.zeros(13)
    x[0:3] = p; x[3] = 1.0; x[7:10] = v
    return x


def _hover_nominal(p, B, N):
    return np.full((B, N, 4), hover_thrust(p), dtype=np.float32)


def cfg0(K=256, N=20) -> Workload:
    """Tiny gate-progress MPPI (BASELINE.json configs[0])."""
    p = base_params(K=K, N=N, B=1, objective=OBJ_GATE, sigma=1.0)
    p["lambda"] = _f32(1.0)
    x0 = _level_state((5.0, -2.0, 1.5))[None].astype(np.float32)
    return Workload("cfg0_gate_tiny", p, x0, np.zeros(1, np.int32), _hover_nominal(p, 1, N),
                    gates=circle_gates(), seed=0, iters=1)


def cfg1(K=4096, N=50, iters=10) -> Workload:
    """Gate progress at real-time scale, 10 warm-started iterations (configs[1])."""
    p = base_params(K=K, N=N, B=1, objective=OBJ_GATE, sigma=1.5)
    p["lambda"] = _f32(0.5)
    gates = lemniscate_gates()
    c0 = gates[0, 0:3].astype(np.float64); n0 = gates[0, 3:6].astype(np.float64)
    x0 = _level_state(c0 - 3.0 * n0, 3.0 * n0)[None].astype(np.float32)
    return Workload("cfg1_gate_K4096_N50", p, x0, np.zeros(1, np.int32), _hover_nominal(p, 1, N),
                    gates=gates, seed=0, iters=iters)


def cfg2(K=4096, N=50, extra_rows=0) -> Workload:
    """Trajectory tracking on a Lissajous reference (configs[2]); x0 = ref[0]  [R-15]."""
    p = base_params(K=K, N=N, B=1, objective=OBJ_TRACK, sigma=1.5)
    p["lambda"] = _f32(0.5)
    ref = lissajous_reference(N + 1 + extra_rows, p["dt"], p["g"])
    x0 = ref[0:1].copy()
    return Workload("cfg2_track_K4096_N50", p, x0, np.zeros(1, np.int32), _hover_nominal(p, 1, N),
                    ref=ref, seed=0, iters=1)


def cfg3(K=8192, N=50) -> Workload:
    """Contouring on a 500-point spline path through the circle-track gate centres (configs[3])."""
    p = base_params(K=K, N=N, B=1, objective=OBJ_CONTOUR, sigma=1.5)
    p["lambda"] = _f32(0.5)
    path = spline_path(circle_gates()[:, 0:3], 500)
    x0 = _level_state((5.0, -2.0, 1.5))[None].astype(np.float32)
    return Workload("cfg3_contour_K8192_N50", p, x0, np.full(1, -1, np.int32),
                    _hover_nominal(p, 1, N), path=path, closed=True, seed=0, iters=1)


def cfg4(K=4096, N=50, B=64, steps=500) -> Workload:
    """Batched closed loop: B jittered drones on the circle track (configs[4])."""
    p = base_params(K=K, N=N, B=B, objective=OBJ_GATE, sigma=1.5)
    p["lambda"] = _f32(0.5)
    rng = np.random.default_rng(7)
    x0 = np.tile(_level_state((5.0, -2.0, 1.5)), (B, 1))
    x0[:, 0:3] += rng.uniform(-0.5, 0.5, (B, 3))
    x0[:, 7:10] += rng.uniform(-1.0, 1.0, (B, 3))
    return Workload(f"cfg4_gate_closed_loop_B{B}", p, x0.astype(np.float32),
                    np.zeros(B, np.int32), _hover_nominal(p, B, N), gates=circle_gates(), seed=0,
                    iters=steps)


def stress_gate(K=1024, N=30) -> Workload:
    """Crossing-heavy case: 3 m before gate 0 at 6 m/s, offset towards a corner
    of the opening, sigma 1.5, so that about two thirds of the samples pass and one third miss:
    the pass / miss / switch branches are all exercised at scale."""
    p = base_params(K=K, N=N, B=1, objective=OBJ_GATE, sigma=1.5)
    p["lambda"] = _f32(0.5)
    gates = circle_gates()
    c0 = gates[0, 0:3].astype(np.float64); n0 = gates[0, 3:6].astype(np.float64)
    h0 = gates[0, 6:9].astype(np.float64)
    x0 = _level_state(c0 - 3.0 * n0 + 0.55 * h0 + np.array([0, 0, 0.5]), 6.0 * n0)
    return Workload("stress_gate_crossings", p, x0[None].astype(np.float32),
                    np.zeros(1, np.int32), _hover_nominal(p, 1, N), gates=gates, seed=3, iters=1)


def gate_paper(K=4096, N=50) -> Workload:
    """The paper's own J_gate (eq.(6),(7) + temporal check) on the
    configs[1] track: squared-distance progress, Q_near = 2 inside r_near = 1.5 m (the paper gives
    neither value), no pass bonus / miss penalty, all states of the previous iteration in front."""
    wl = cfg1(K=K, N=N, iters=1)
    p = dict(wl.params, objective=OBJ_GATE_PAPER, gate_pass_bonus=0.0, gate_miss_penalty=0.0,
             q_near=_f32(2.0), r_near=_f32(1.5))
    return Workload(f"gate_paper_K{K}_N{N}", p, wl.x0, wl.start, wl.u_nom, gates=wl.gates, seed=wl.seed)


def stress_gate_paper(K=1024, N=30, flag_seed=5) -> Workload:
    """stress_gate under the paper's J_gate with random previous-iteration flags, so that registered and
    unregistered passes, misses and the near term all occur at scale."""
    wl = stress_gate(K=K, N=N)
    p = dict(wl.params, objective=OBJ_GATE_PAPER, q_near=_f32(2.0), r_near=_f32(1.5))
    rng = np.random.default_rng(flag_seed)
    front = (rng.uniform(size=(1, N + 1)) < 0.6).astype(np.int32)
    return Workload("stress_gate_paper", p, wl.x0, wl.start, wl.u_nom, gates=wl.gates, seed=wl.seed,
                    prev_front=front)


def _rate_model(wl: Workload, name: str, **over) -> Workload:
    """The same scene under the paper's own input model (Table I PAPER.md:216-221;
    SURVEY.md NEXT-2): u = thrust RATES with the four rotor thrusts as extra states (x0 gets T = hover),
    rates clamped to +-10 N/s, thrusts to [0, 10] N, sigma 5 N/s, rotor drag D = diag(0.25, 0.25, 0.1) 1/s
    and a soft body-rate limit at 10 rad/s (the paper prints no drag value and no penalty form)."""
    p = dict(wl.params, input_model=1, rate_max=_f32(10.0), T_max=_f32(10.0), sigma=_f32(5.0),
             drag_x=_f32(0.25), drag_y=_f32(0.25), drag_z=_f32(0.1), w_limit=_f32(1.0), omega_max=_f32(10.0))
    p.update(over)
    B = wl.x0.shape[0]
    x0 = np.concatenate([wl.x0, np.full((B, 4), hover_thrust(p), np.float32)], axis=1)
    return Workload(name, p, x0.astype(np.float32), wl.start, np.zeros_like(wl.u_nom), gates=wl.gates,
                    ref=wl.ref, path=wl.path, closed=wl.closed, seed=wl.seed, prev_front=wl.prev_front)


def rate_gate_paper(K=4096, N=50) -> Workload:
    """NEXT-2 + NEXT-1 together: the paper's model and the paper's J_gate on the configs[1] track."""
    return _rate_model(gate_paper(K=K, N=N), f"rate_gate_paper_K{K}_N{N}")


def rate_track(K=4096, N=50) -> Workload:
    """NEXT-2 under the tracking objective: eq.(8)'s input term acts on the rates."""
    return _rate_model(cfg2(K=K, N=N), f"rate_track_K{K}_N{N}")


def rate_stress(K=1024, N=30) -> Workload:
    """Crossing-heavy gate case (objective 0) under the rate model, with faster noise so that the rate
    clamp acts on ~10 % of the draws and thrusts reach their range (much faster and the explicit RK4
    itself goes unstable on the tumbling samples: |omega| dt > 2.8, costs beyond fp32 range)."""
    return _rate_model(stress_gate(K=K, N=N), "rate_stress_gate", sigma=_f32(12.0), rate_max=_f32(20.0))


def contour_paper(K=4096, N=50) -> Workload:
    """The paper's own contouring formulation (eq.(9)) on configs[3]'s
    spline path under the paper's input model: states + (theta, v_theta), sampled inputs = four thrust
    rates + the progress acceleration (sigma_v 5 m/s^2, range +-20, v_theta in [0, 10]: Table I), weights
    q_c 200, q_l 50, mu 2 (configs[3]), r_dv 0.01, R 0.01 on the rates.  theta_0 = arc length of the path
    vertex nearest to p_0, v_theta,0 = 2 m/s."""
    wl = _rate_model(cfg3(K=K, N=N), f"contour_paper_K{K}_N{N}", objective=OBJ_CONTOUR_PAPER, sigma_v=_f32(5.0),
                     dv_max=_f32(20.0), v_theta_max=_f32(10.0), r_dv=_f32(0.01))
    pts = wl.path.astype(np.float64)
    s = np.concatenate([[0.0], np.cumsum(np.linalg.norm(np.diff(pts, axis=0), axis=1))])
    i = int(np.argmin(np.sum((pts - wl.x0[0, 0:3].astype(np.float64)) ** 2, axis=1)))
    x0 = np.concatenate([wl.x0, np.array([[s[i], 2.0]], np.float32)], axis=1).astype(np.float32)
    wl.x0 = x0
    wl.v_nom = np.zeros((1, N), np.float32)
    return wl


def figure8_start(B, rng, jitter=0.2):
    """B jittered start states 3 m before gate 0 of the configs[1] lemniscate, flying at 3 m/s towards it [R-16]."""
    gates = lemniscate_gates()
    c0 = gates[0, 0:3].astype(np.float64); n0 = gates[0, 3:6].astype(np.float64)
    x0 = np.tile(_level_state(c0 - 3.0 * n0, 3.0 * n0), (B, 1))
    x0[:, 0:3] += rng.uniform(-jitter, jitter, (B, 3))
    return gates, x0.astype(np.float32)


def lap(kind="gate", B=8, K=4096, N=50, steps=1500, track="circle") -> Workload:
    """Closed-loop lap experiment (shaped like Table II) on the 4-gate
    circle of configs[0] / its spline path / the Lissajous reference, or (track = "figure8": the stand-in for
    the paper's Figure-8 track) on the 7-gate lemniscate of configs[1] with gate heights 1-3 m / the
    spline path through its gate centres; B jittered drones.  The noise and
    temperature are the ones a controller can actually fly with -- sigma 0.5 N, lambda 0.02, w_omega
    0.001: under configs[4]'s sigma 1.5 / lambda 0.5 the closed loop does not stay in the air (measured)."""
    rng = np.random.default_rng(7)
    tune = dict(sigma=_f32(0.5), w_omega=_f32(0.001))
    if track not in ("circle", "figure8"):
        raise ValueError("track must be 'circle' or 'figure8'")
    if kind in ("track",) and track != "circle":
        raise ValueError("the tracking lap flies the Lissajous reference: track = 'circle' only")
    if kind in ("gate", "gate_paper"):
        wl = cfg4(K=K, N=N, B=B, steps=steps)
        if track == "figure8":
            wl.gates, wl.x0 = figure8_start(B, rng)
        p = dict(wl.params, **tune)
        if kind == "gate_paper":
            p.update(objective=OBJ_GATE_PAPER, gate_pass_bonus=0.0, gate_miss_penalty=0.0, q_near=_f32(0.5), r_near=_f32(1.5))
        p["lambda"] = _f32(0.5 if kind == "gate_paper" else 0.02)      # squared distances: larger cost scale
        return Workload(f"lap_{kind}_{track}_B{B}", p, wl.x0, wl.start, wl.u_nom, gates=wl.gates, seed=0, iters=steps)
    if kind == "contour_paper":
        # the paper's own contouring under the paper's model; tuned like the other lap workloads so that it flies
        base = contour_paper(K=K, N=N)
        if track == "figure8":                 # spline path through the lemniscate's gate centres, start on it
            gates, x13 = figure8_start(1, np.random.default_rng(0), 0.0)
            base.path = spline_path(gates[:, 0:3], 500)
            pts = base.path.astype(np.float64)
            s = np.concatenate([[0.0], np.cumsum(np.linalg.norm(np.diff(pts, axis=0), axis=1))])
            i = int(np.argmin(np.sum((pts - x13[0, 0:3].astype(np.float64)) ** 2, axis=1)))
            base.x0 = np.concatenate([x13, base.x0[:, 13:17], np.array([[s[i], 3.0]], np.float32)], axis=1).astype(np.float32)
        p = dict(base.params, B=B, sigma=_f32(3.0), sigma_v=_f32(3.0), w_omega=_f32(0.001), q_contour=_f32(200.0),
                 q_lag=_f32(100.0), mu_progress=_f32(10.0))
        p["lambda"] = _f32(1.0)
        x0 = np.repeat(base.x0, B, 0)
        x0[:, 0:3] += rng.uniform(-0.2, 0.2, (B, 3)).astype(np.float32)
        return Workload(f"lap_{kind}_{track}_B{B}", p, x0.astype(np.float32), np.repeat(base.start, B, 0), np.repeat(base.u_nom, B, 0),
                        path=base.path, closed=base.closed, v_nom=np.repeat(base.v_nom, B, 0), seed=0, iters=steps)
    base = cfg2(K=K, N=N, extra_rows=steps + 1) if kind == "track" else cfg3(K=K, N=N)
    if kind == "contour" and track == "figure8":
        gates, x13 = figure8_start(1, np.random.default_rng(0), 0.0)
        base.path = spline_path(gates[:, 0:3], 500)
        base.x0 = x13
    p = dict(base.params, B=B, **tune)
    p["lambda"] = _f32(0.02 if kind == "contour" else 0.5)
    x0 = np.repeat(base.x0, B, 0)
    x0[:, 0:3] += rng.uniform(-0.2, 0.2, (B, 3)).astype(np.float32)
    return Workload(f"lap_{kind}_B{B}", p, x0.astype(np.float32), np.repeat(base.start, B, 0),
                    np.repeat(base.u_nom, B, 0), ref=base.ref, path=base.path, closed=base.closed, seed=0, iters=steps)


def table1(kind="gate") -> Workload:
    """The sizes of the paper's own Table I: M = 8192 samples, horizon K = 20 steps of
    dt = 0.03 s, lambda = 0.01, thrust-rate inputs in [-10, 10] N/s, thrusts in [0, 10] N, body rates limited
    to 10 rad/s, (contouring) progress acceleration in [-20, 20], v_theta in [0, 10] -- on the synthetic circle
    track / its spline path, under the paper's J_gate ("gate") or the paper's contouring ("contour")."""
    wl = rate_gate_paper(K=8192, N=20) if kind == "gate" else contour_paper(K=8192, N=20)
    wl.params.update(dt=_f32(0.03))
    wl.params["lambda"] = _f32(0.01)
    wl.name = f"table1_{kind}_M8192_K20"
    return wl


def replicate(wl: Workload, B: int, jitter: float = 0.0) -> Workload:
    """The same single-controller workload for B controllers (positions jittered by +-jitter m, seeded)."""
    rng = np.random.default_rng(11)
    rep = lambda a: None if a is None else np.repeat(a[:1], B, 0).copy()
    x0 = rep(wl.x0)
    if jitter:
        x0[:, 0:3] += rng.uniform(-jitter, jitter, (B, 3)).astype(np.float32)
    return Workload(f"{wl.name}_x{B}", dict(wl.params, B=B), x0, rep(wl.start), rep(wl.u_nom), gates=wl.gates, ref=wl.ref,
                    path=wl.path, prev_front=rep(wl.prev_front), v_nom=rep(wl.v_nom), closed=wl.closed, seed=wl.seed,
                    iters=wl.iters)


ALL = {"table1_gate": lambda: table1("gate"), "table1_contour": lambda: table1("contour"), "contour_paper": contour_paper, "rate_gate_paper": rate_gate_paper, "rate_track": rate_track, "rate_stress": rate_stress,
       "gate_paper": gate_paper, "stress_gate_paper": stress_gate_paper, "cfg0": cfg0, "cfg1": cfg1, "cfg2": cfg2, "cfg3": cfg3, "cfg4": cfg4,
       "stress_gate": stress_gate}
