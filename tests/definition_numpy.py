"""Independent "definition" evaluator used ONLY to pin the C oracle on tiny inputs (pin P14).

Written separately from oracle/mppi_oracle.c, from the same passages of PAPER.md, in a
different formulation wherever the mathematics allows one: the rotation matrix R(q) is built
in full (eq.(2)), the quaternion kinematics use the 4x4 matrix Lambda(q), torques
come from an allocation matrix, the softmax is scipy's, Philox runs on Python
integers.  A dropped term, wrong sign, or transposed operand in either implementation makes
the two disagree.  It is slow and is never used as an oracle for the GPU path.
"""
from __future__ import annotations

import math

import numpy as np
from scipy.special import softmax

MASK = 0xFFFFFFFF


def philox(ctr, key):
    c = [int(v) & MASK for v in ctr]
    k = [int(v) & MASK for v in key]
    for _ in range(10):
        p0 = 0xD2511F53 * c[0]
        p1 = 0xCD9E8D57 * c[2]
        c = [((p1 >> 32) ^ c[1] ^ k[0]) & MASK, p1 & MASK, ((p0 >> 32) ^ c[3] ^ k[1]) & MASK,
             p0 & MASK]
        k = [(k[0] + 0x9E3779B9) & MASK, (k[1] + 0xBB67AE85) & MASK]
    return c


def normals(seed, k, t, it, b):
    r = philox([k, t, it, b], [seed & MASK, seed >> 32])
    u = [(2 * (w >> 9) + 1) / 2 ** 24 for w in r]
    out = []
    for a, bb in ((u[0], u[1]), (u[2], u[3])):
        rad = math.sqrt(-2.0 * math.log(a))
        out += [rad * math.cos(2 * math.pi * bb), rad * math.sin(2 * math.pi * bb)]
    return np.array(out)


def rot(q):
    w, x, y, z = q
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                     [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                     [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])


def lam(q):
    w, x, y, z = q
    return np.array([[w, -x, -y, -z], [x, w, -z, y], [y, z, w, -x], [z, -y, x, w]])


def fdyn(P, x, T):
    p, q, v, om = x[0:3], x[3:7], x[7:10], x[10:13]
    J = np.diag([P["Jx"], P["Jy"], P["Jz"]])
    l = P["arm"] / math.sqrt(2)
    alloc = np.array([[l, l, -l, -l], [-l, l, l, -l],
                      [P["c_tau"], -P["c_tau"], P["c_tau"], -P["c_tau"]]])
    tau = alloc @ T
    vdot = np.array([0, 0, -P["g"]]) + rot(q) @ np.array([0, 0, np.sum(T)]) / P["mass"]
    qdot = 0.5 * lam(q) @ np.concatenate([[0.0], om])
    omdot = np.linalg.solve(J, tau - np.cross(om, J @ om))
    if any(P.get(k, 0.0) for k in ("drag_x", "drag_y", "drag_z")):
        Dm = np.diag([P["drag_x"], P["drag_y"], P["drag_z"]])          # eq.(2): - R D R^T v
        vdot = vdot - rot(q) @ Dm @ rot(q).T @ v
    return np.concatenate([v, qdot, vdot, omdot])


def rk4(P, x, T):
    h = P["dt"]
    k1 = fdyn(P, x, T); k2 = fdyn(P, x + h / 2 * k1, T)
    k3 = fdyn(P, x + h / 2 * k2, T); k4 = fdyn(P, x + h * k3, T)
    xn = x + h / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
    xn[3:7] /= np.linalg.norm(xn[3:7])
    return xn


def rk4_rate(P, x, u):
    """17-state thrust-rate model: z = [x13, T4], z' = [f_dyn(x13, T), u]."""
    h = P["dt"]
    f = lambda z: np.concatenate([fdyn(P, z[:13], z[13:]), u])
    k1 = f(x); k2 = f(x + h / 2 * k1); k3 = f(x + h / 2 * k2); k4 = f(x + h * k3)
    xn = x + h / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
    xn[3:7] /= np.linalg.norm(xn[3:7])
    xn[13:] = np.clip(xn[13:], P["T_min"], P["T_max"])
    return xn


def path_tables(pts, closed):
    n = len(pts)
    seg = np.linalg.norm(np.diff(pts, axis=0), axis=1)
    s = np.concatenate([[0.0], np.cumsum(seg)])
    L = s[-1] + (np.linalg.norm(pts[0] - pts[-1]) if closed else 0.0)
    if closed:
        d = np.roll(pts, -1, axis=0) - np.roll(pts, 1, axis=0)
    else:
        d = np.empty_like(pts)
        d[1:-1] = pts[2:] - pts[:-2]; d[0] = pts[1] - pts[0]; d[-1] = pts[-1] - pts[-2]
    return s, d / np.linalg.norm(d, axis=1, keepdims=True), L


def nearest(pts, closed, p, centre, W):
    n = len(pts)
    idx = np.arange(n) if centre < 0 else np.arange(centre - W, centre + W + 1)
    if closed:
        idx = idx % n
    else:
        idx = idx[(idx >= 0) & (idx < n)]
    d2 = np.sum((pts[idx] - p) ** 2, axis=1)
    return int(idx[int(np.argmin(d2))])


def path_eval(pts, closed, theta):
    """P(theta) and unit tangent by linear interpolation over the (closed) polyline, written with
    searchsorted on an explicitly extended table -- a different route from the oracle's scan."""
    s, tan, L = path_tables(pts, closed)
    if closed:
        th = theta % L
        se = np.concatenate([s, [L]]); pe = np.vstack([pts, pts[:1]]); te = np.vstack([tan, tan[:1]])
    else:
        th = min(max(theta, 0.0), s[-1]); se, pe, te = s, pts, tan
    i = int(np.searchsorted(se, th, side="right")) - 1
    i = min(max(i, 0), len(se) - 2)
    lam = (th - se[i]) / (se[i + 1] - se[i])
    t = (1 - lam) * te[i] + lam * te[i + 1]
    return (1 - lam) * pe[i] + lam * pe[i + 1], t / np.linalg.norm(t)


def rollout_cost5(P, trk, x0, u_nom, v_nom, seed, it, k, b):
    """Objective 4 (the paper's eq.(9)): -> (J, du[N,4], dv[N])"""
    N, h = P["N"], P["dt"]
    x = np.array(x0, dtype=float)
    J = 0.0; du = np.zeros((N, 4)); dvs = np.zeros(N)
    for t in range(N):
        u = np.clip(u_nom[t] + P["sigma"] * normals(seed, k, t, it, b), -P["rate_max"], P["rate_max"])
        z5 = normals(seed, k, t + 2 ** 31, it, b)[0]
        dv = float(np.clip(v_nom[t] + P["sigma_v"] * z5, -P["dv_max"], P["dv_max"]))
        du[t] = u - u_nom[t]; dvs[t] = dv - v_nom[t]
        pos, tg = path_eval(trk["path"], trk["closed"], x[17])
        e = x[0:3] - pos
        el = e @ tg
        J += (P["q_lag"] * el ** 2 + P["q_contour"] * max(e @ e - el ** 2, 0.0) + P["w_omega"] * np.sum(x[10:13] ** 2)
              + P["r_dv"] * dv ** 2 + P["R"] * np.sum(u ** 2) - P["mu_progress"] * x[18])
        xn = np.empty(19)
        xn[:17] = rk4_rate(P, x[:17], u)
        xn[17] = x[17] + h * x[18] + 0.5 * h * h * dv
        xn[18] = min(max(x[18] + h * dv, 0.0), P["v_theta_max"])
        J += P["w_limit"] * np.sum(np.maximum(np.abs(xn[10:13]) - P["omega_max"], 0.0) ** 2)
        x = xn
    return J, du, dvs


def mppi_step5(P, trk, x0, u_nom, v_nom, seed, it, b=0):
    res = [rollout_cost5(P, trk, x0, u_nom, v_nom, seed, it, k, b) for k in range(P["K"])]
    J = np.array([r[0] for r in res]); du = np.array([r[1] for r in res]); dv = np.array([r[2] for r in res])
    w = softmax(-J / P["lambda"])
    return J, w, u_nom + np.einsum("k,ktn->tn", w, du), v_nom + w @ dv, du, dv


def rollout_cost(P, trk, x0, start, u_nom, seed, it, k, b):
    """-> (J, du[N,4], final aux)"""
    N = P["N"]
    hover = P["mass"] * P["g"] / 4
    xs = [np.array(x0, dtype=float)]
    Ts = []
    rate = P.get("input_model", 0) == 1
    lo, hi = (-P["rate_max"], P["rate_max"]) if rate else (P["T_min"], P["T_max"])
    for t in range(N):
        T = np.clip(u_nom[t] + P["sigma"] * normals(seed, k, t, it, b), lo, hi)
        Ts.append(T)
        xs.append(rk4_rate(P, xs[-1], T) if rate else rk4(P, xs[-1], T))
    Ts = np.array(Ts)
    du = Ts - u_nom
    J = 0.0
    if rate:                                   # soft body-rate limit on every post-step state
        for t in range(1, N + 1):
            J += P["w_limit"] * np.sum(np.maximum(np.abs(xs[t][10:13]) - P["omega_max"], 0.0) ** 2)
    aux = start
    if P["objective"] == 0:
        gates = trk["gates"]
        for t in range(N):
            g = gates[aux]
            c, n, h, aw, ah = g[0:3], g[3:6], g[6:9], g[9], g[10]
            a, bpt = xs[t][0:3], xs[t + 1][0:3]
            J += np.linalg.norm(bpt - c) - np.linalg.norm(a - c)
            J += P["w_omega"] * np.sum(xs[t + 1][10:13] ** 2)
            sa, sb = n @ (a - c), n @ (bpt - c)
            if sa < 0 <= sb:
                hit = a + (bpt - a) * (sa / (sa - sb)) - c
                if abs(h @ hit) <= aw and abs(np.cross(h, n) @ hit) <= ah:
                    J -= P["gate_pass_bonus"]; aux = (aux + 1) % len(gates)
                else:
                    J += P["gate_miss_penalty"]
    elif P["objective"] == 3:
        # the paper's own J_gate: eq.(6),(7) PAPER.md:105-129 + the temporal check of Fig. 2
        gates = trk["gates"]
        front = trk.get("prev_front")
        aux = start % len(gates)
        g0 = aux
        for t in range(N):
            g = gates[aux]
            c, n, h, aw, ah = g[0:3], g[3:6], g[6:9], g[9], g[10]
            a, bpt = xs[t][0:3], xs[t + 1][0:3]
            J += np.sum((bpt - c) ** 2) - np.sum((a - c) ** 2)
            cn = gates[g0][0:3] if P.get("near_mode", 0) == 1 else c        # eq.(7): start gate of the horizon, or own target
            if np.linalg.norm(a - cn) < P["r_near"]:
                J += P["q_near"] * np.sum((a - cn) ** 2)
            J += P["w_omega"] * np.sum(xs[t + 1][10:13] ** 2)
            sa, sb = n @ (a - c), n @ (bpt - c)
            if sa < 0 <= sb:
                hit = a + (bpt - a) * (sa / (sa - sb)) - c
                if abs(h @ hit) <= aw and abs(np.cross(h, n) @ hit) <= ah:
                    if aux != g0 or front is None or front[b][t + 1]:
                        J -= P["gate_pass_bonus"]; aux = (aux + 1) % len(gates)
                else:
                    J += P["gate_miss_penalty"]
    elif P["objective"] == 1:
        ref = trk["ref"]
        Q = np.diag([P["Qp"]] * 3 + [P["Qv"]] * 3 + [P["Qw"]] * 3)
        for t in range(N + 1):
            x, r = xs[t], ref[start + t]
            e = np.concatenate([x[0:3] - r[0:3], x[7:10] - r[7:10], x[10:13] - r[10:13]])
            qerr = x[3:7] @ x[3:7] + r[3:7] @ r[3:7] - 2 * abs(x[3:7] @ r[3:7])
            J += e @ Q @ e + P["Qq"] * qerr
            if t < N:
                J += P["R"] * np.sum((Ts[t] - (0.0 if rate else hover)) ** 2)
    else:
        pts, closed, W = trk["path"], trk["closed"], P["window"]
        s, tan, L = path_tables(pts, closed)
        aux = nearest(pts, closed, xs[0][0:3], start, W)
        th_prev = s[aux] + (xs[0][0:3] - pts[aux]) @ tan[aux]
        for t in range(1, N + 1):
            p = xs[t][0:3]
            aux = nearest(pts, closed, p, aux, W)
            e = p - pts[aux]
            el = e @ tan[aux]
            ec2 = max(e @ e - el * el, 0.0)
            th = s[aux] + el
            d = th - th_prev
            if closed:
                d -= L * math.ceil((d - L / 2) / L)      # into (-L/2, L/2]
            J += P["q_contour"] * ec2 + P["q_lag"] * el * el - P["mu_progress"] * d
            J += P["w_omega"] * np.sum(xs[t][10:13] ** 2)
            th_prev = th
    return J, du, aux


def mppi_step(P, trk, x0, start, u_nom, seed, it, b=0):
    K = P["K"]
    res = [rollout_cost(P, trk, x0, start, u_nom, seed, it, k, b) for k in range(K)]
    J = np.array([r[0] for r in res]); du = np.array([r[1] for r in res])
    w = softmax(-J / P["lambda"])
    return J, w, u_nom + np.einsum("k,ktn->tn", w, du), du
