"""Closed-loop lap experiment shaped like the paper's Table II:
the controller (mppi_step, one or more iterations per control step) flies the plant (mppi_sim_step,
the same RK4 model) around a synthetic track; the flight is logged on the device and reduced on the
host to the quantities the paper tabulates -- flight time for a number of laps, distance to the gate
centre at every pass ("waypoint distance"), tracking RMSE -- plus speed statistics.

The paper's own tracks, CPC references and numbers are not available,
so these metrics describe the synthetic tracks of workloads.py and cannot be compared with Table II.

Everything numerical on the flight path runs in libmppi's kernels; this module only drives the loop
(argument marshalling through binding.Mppi) and post-processes the logged states in float64 numpy.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass
class FlightLog:
    x: np.ndarray          # [steps + 1, B, xdim] float32: plant state before every control step + the last
                           # (xdim 13; 17 under the rate model; 19 under objective 4: ..., theta, v_theta)
    start: np.ndarray      # [steps + 1, B] int32: the controller's start index (target gate / row / path index)
    dt: float


def fly(m, wl, steps: int, iters_per_step: int = 1, seed=None, prev_front_feedback: bool = False) -> FlightLog:
    """Runs `steps` control steps of the closed loop on the GPU and returns the logged plant states.
    m: binding.Mppi created from wl.params with its track set.  One control step = `iters_per_step`
    warm-started MPPI iterations (Philox iter = step * iters_per_step + j), then the plant step with
    u_new[0], the start-index advance and the one-step shift of the nominal [R-14].  With
    prev_front_feedback (objective 3) the "in front" flags of each new nominal, shifted by one control
    step, are fed to the next step (Fig. 2)."""
    import torch
    seed = wl.seed if seed is None else seed
    dev = torch.device("cuda", torch.cuda.current_device())
    x = torch.from_numpy(np.ascontiguousarray(wl.x0)).to(dev)
    start = torch.from_numpy(np.ascontiguousarray(wl.start)).to(dev)
    u = torch.from_numpy(np.ascontiguousarray(wl.u_nom)).to(dev)
    B, K = m.B, m.K
    cost = torch.empty((B, K), device=dev); w = torch.empty_like(cost)
    log_x = torch.empty((steps + 1, B, x.shape[1]), device=dev)
    log_s = torch.empty((steps + 1, B), dtype=torch.int32, device=dev)
    front = None
    progress = m.params.objective == 4        # the paper's contouring: rows of 19, fifth column v [B,N]
    if progress:
        v = torch.from_numpy(np.ascontiguousarray(wl.v_nom)).to(dev)
        m.set_progress(v)                     # in place
    for i in range(steps):
        log_x[i].copy_(x); log_s[i].copy_(start)
        if progress:
            for j in range(iters_per_step):
                m.step(x, start, u, seed, i * iters_per_step + j, u_new=u, cost=cost, weights=w)
            m.sim_step_progress(x, u, v)
            continue
        if prev_front_feedback:
            m.set_prev_front(front)
        for j in range(iters_per_step):
            m.step(x, start, u, seed, i * iters_per_step + j, u_new=u, cost=cost, weights=w)
        if prev_front_feedback:
            f = m.front_flags(x, start, u)
            front = torch.cat([f[:, 1:], f[:, -1:]], dim=1).contiguous()
        m.sim_step(x, start, u, u_nom_next=u)
    log_x[steps].copy_(x); log_s[steps].copy_(start)
    torch.cuda.synchronize()
    return FlightLog(log_x.cpu().numpy(), log_s.cpu().numpy(), float(wl.params["dt"]))


# ---- host-side reduction of a flight log (float64) ------------------------------------------------------

def gate_passes(p: np.ndarray, gates: np.ndarray, first_gate: int = 0):
    """Valid gate passes of ONE flown position sequence p [T, 3] through the gates in order, by the
    geometric rule of [R-9]: segment p_t -> p_{t+1} crosses the current gate's plane front to back
    inside the opening.  -> list of (step index t+1, gate index, distance of the crossing point from the
    gate centre, interpolation fraction alpha)."""
    p = np.asarray(p, np.float64); gates = np.asarray(gates, np.float64)
    G = gates.shape[0]
    g = first_gate % G
    out = []
    for t in range(len(p) - 1):
        c, n, h, ah, av = gates[g, 0:3], gates[g, 3:6], gates[g, 6:9], gates[g, 9], gates[g, 10]
        s0, s1 = n @ (p[t] - c), n @ (p[t + 1] - c)
        if s0 < 0.0 <= s1:
            a = s0 / (s0 - s1)
            hit = p[t] + a * (p[t + 1] - p[t]) - c
            if abs(h @ hit) <= ah and abs(np.cross(h, n) @ hit) <= av:
                out.append((t + 1, g, float(np.linalg.norm(hit)), float(a)))
                g = (g + 1) % G
    return out


def lap_metrics(log: FlightLog, gates: np.ndarray, laps: int, first_gate: int = 0) -> list[dict]:
    """Per drone: flight time for `laps` laps (time of the laps*G-th valid pass, None if not reached),
    passes made, waypoint distances (min / mean / max over the counted passes), mean and top speed."""
    G = gates.shape[0]
    res = []
    for b in range(log.x.shape[1]):
        p = log.x[:, b, 0:3].astype(np.float64)
        passes = gate_passes(p, gates, first_gate)
        need = laps * G
        counted = passes[:need]
        t_done = None
        if len(passes) >= need:
            t1, _, _, a = passes[need - 1]
            t_done = (t1 - 1 + a) * log.dt
        d = np.array([q[2] for q in counted])
        n_flown = passes[need - 1][0] if t_done is not None else len(p) - 1
        speed = np.linalg.norm(log.x[: n_flown + 1, b, 7:10].astype(np.float64), axis=1)
        nan = float("nan")
        res.append(dict(passes=len(passes), flight_time_s=t_done, wp_dist_min=float(d.min()) if d.size else nan,
                        wp_dist_mean=float(d.mean()) if d.size else nan, wp_dist_max=float(d.max()) if d.size else nan,
                        speed_mean=float(speed.mean()), speed_max=float(speed.max())))
    return res


def tracking_rmse(log: FlightLog, ref: np.ndarray, first_row: int = 0) -> np.ndarray:
    """Per drone: RMS position error between the flown states and the reference rows they were flown
    against (row first_row + step; one row per dt)."""
    T = log.x.shape[0]
    r = np.asarray(ref, np.float64)[first_row: first_row + T, 0:3]
    e = log.x[: len(r), :, 0:3].astype(np.float64) - r[:, None, :]
    return np.sqrt((e ** 2).sum(-1).mean(0))


def progress_metrics(log: FlightLog, path: np.ndarray) -> list[dict]:
    """Objective 4 (rows of 19): per drone the progress made (theta_end - theta_0, in laps of the closed path
    too), the time of every completed lap of theta, the largest distance between the drone and P(theta)
    (how well the virtual progress state and the vehicle stay together) and speed statistics."""
    P = np.asarray(path, np.float64)
    seg = np.linalg.norm(np.diff(np.vstack([P, P[:1]]), axis=0), axis=1)
    s = np.concatenate([[0.0], np.cumsum(seg)])                # s[P] = L
    L = float(s[-1])
    Pc = np.vstack([P, P[:1]])
    res = []
    for b in range(log.x.shape[1]):
        th = log.x[:, b, 17].astype(np.float64)
        p = log.x[:, b, 0:3].astype(np.float64)
        tw = np.mod(th, L)
        on = np.stack([np.interp(tw, s, Pc[:, a]) for a in range(3)], axis=1)
        adv = th - th[0]
        lap_t = [float(np.argmax(adv >= k * L) * log.dt) for k in range(1, int(adv[-1] // L) + 1)]
        speed = np.linalg.norm(log.x[:, b, 7:10].astype(np.float64), axis=1)
        res.append(dict(progress_m=float(adv[-1]), laps=float(adv[-1] / L), lap_times_s=lap_t,
                        dist_to_progress_point_max=float(np.linalg.norm(p - on, axis=1).max()),
                        speed_mean=float(speed.mean()), speed_max=float(speed.max())))
    return res


def contour_rms(log: FlightLog, path: np.ndarray) -> np.ndarray:
    """Per drone: RMS distance of the flown positions from the (densely sampled, closed) path polyline."""
    P = np.asarray(path, np.float64)
    A, Bp = P, np.roll(P, -1, axis=0)
    d = Bp - A
    dd = (d ** 2).sum(-1)
    out = []
    for b in range(log.x.shape[1]):
        p = log.x[:, b, 0:3].astype(np.float64)
        t = np.clip(((p[:, None, :] - A[None]) * d[None]).sum(-1) / dd[None], 0.0, 1.0)
        q = A[None] + t[..., None] * d[None]
        dist2 = ((p[:, None, :] - q) ** 2).sum(-1).min(1)
        out.append(np.sqrt(dist2.mean()))
    return np.array(out)


# ---- the experiment as a command: python -m paper_2509_14726_b200.closed_loop [--track circle|figure8] ---------------

def run_table(track: str = "circle", B: int = 8, K: int = 4096, laps: int = 3, horizon_s: float = 40.0):
    """Flies every objective on one synthetic track and prints the rows of DESIGN.md section 10's table (markdown).
    Not comparable with the paper's Table II: its tracks and references are not available."""
    import time
    import torch
    from . import binding as Bd
    from . import workloads as W
    rows = [("gate", 1), ("gate", 2), ("gate_paper", 1), ("gate_paper", 2), ("contour", 1), ("contour_paper", 1), ("contour_paper", 2)]
    if track == "circle":
        rows.insert(4, ("track", 1))
    print(f"| track | objective | iterations / control step | GPU time / control step | drones finishing {laps} laps in {horizon_s:.0f} s | "
          "flight time (s) | waypoint distance mean / max (m) | mean / top speed (m/s) | other |")
    print("|---|---|---|---|---|---|---|---|---|")
    for kind, iters in rows:
        wl = W.lap(kind, B=B, K=K, track=track)
        steps = int(round(horizon_s / wl.params["dt"]))
        if kind == "track":
            wl = W.lap(kind, B=B, K=K, steps=steps, track=track)
        m = Bd.Mppi(wl.params)
        m.set_track(wl)
        fly(m, wl, 20, iters_per_step=iters, prev_front_feedback=(kind == "gate_paper"))          # warm-up
        torch.cuda.synchronize(); t0 = time.perf_counter()
        log = fly(m, wl, steps, iters_per_step=iters, prev_front_feedback=(kind == "gate_paper"))
        us = (time.perf_counter() - t0) / steps * 1e6
        m.close()
        if kind in ("gate", "gate_paper"):
            mt = lap_metrics(log, wl.gates, laps=laps)
            done = [q for q in mt if q["flight_time_s"] is not None]
            ft = f"{min(q['flight_time_s'] for q in done):.1f} - {max(q['flight_time_s'] for q in done):.1f}" if done else "-"
            wp = (f"{np.mean([q['wp_dist_mean'] for q in done]):.2f} / {max(q['wp_dist_max'] for q in done):.2f}" if done else "-")
            sp = f"{np.mean([q['speed_mean'] for q in mt]):.1f} / {max(q['speed_max'] for q in mt):.1f}"
            print(f"| {track} | {kind} | {iters} | {us:.0f} us | {len(done)} / {B} | {ft} | {wp} | {sp} | passes {min(q['passes'] for q in mt)} - {max(q['passes'] for q in mt)} |", flush=True)
        elif kind == "track":
            e = tracking_rmse(log, wl.ref)
            print(f"| {track} | tracking (Lissajous reference) | {iters} | {us:.0f} us | - | - | - | - | position RMSE {e.min():.2f} - {e.max():.2f} m |", flush=True)
        elif kind == "contour":
            e = contour_rms(log, wl.path)
            sp = np.linalg.norm(log.x[:, :, 7:10].astype(np.float64), axis=-1)
            print(f"| {track} | contouring (search) | {iters} | {us:.0f} us | - | - | - | {sp.mean():.1f} / {sp.max():.1f} | contour RMS {e.min():.2f} - {e.max():.2f} m |", flush=True)
        else:
            pm = progress_metrics(log, wl.path)
            e = contour_rms(log, wl.path)
            done = [q for q in pm if len(q["lap_times_s"]) >= laps]
            ft = f"{min(q['lap_times_s'][laps - 1] for q in done):.1f} - {max(q['lap_times_s'][laps - 1] for q in done):.1f}" if done else "-"
            print(f"| {track} | the paper's contouring, eq.(9) | {iters} | {us:.0f} us | {len(done)} / {B} (laps of theta) | {ft} | - | "
                  f"{np.mean([q['speed_mean'] for q in pm]):.1f} / {max(q['speed_max'] for q in pm):.1f} | contour RMS {e.min():.2f} - {e.max():.2f} m; "
                  f"vehicle <= {max(q['dist_to_progress_point_max'] for q in pm):.2f} m from P(theta); laps {min(q['laps'] for q in pm):.1f} - {max(q['laps'] for q in pm):.1f} |", flush=True)


if __name__ == "__main__":
    import argparse
    ap = argparse.ArgumentParser(description="closed-loop lap experiment on the synthetic tracks (DESIGN.md section 10)")
    ap.add_argument("--track", default="circle", choices=["circle", "figure8"])
    ap.add_argument("--drones", type=int, default=8)
    ap.add_argument("--samples", type=int, default=4096)
    ap.add_argument("--laps", type=int, default=3)
    ap.add_argument("--seconds", type=float, default=40.0)
    a = ap.parse_args()
    run_table(a.track, a.drones, a.samples, a.laps, a.seconds)
