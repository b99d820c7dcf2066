"""The mathematics behind the time-parallel kernel (csrc/mppi_scan.cuh), checked on the CPU against the oracle's
sequential RK4 (oracle.rk4_step, eq.(2) PAPER.md:65-72 + per-step renormalisation [R-5]).

The kernel claims that, with the thrusts given and Jx == Jy, one RK4 rollout is a cascade of linear recurrences that can
be cut into chunks, each integrated from a neutral start, and joined exactly:
  omega_z   a prefix sum;
  omega_xy  one RK4 step is a complex affine map  w -> H w + p  (H from a homogeneous run, p from a particular run);
  q         one RK4 step is  q -> q (x) m,  renormalisation commutes with the products;
  v, p      sums of thrust directions, carried from the chunk's own frame into the world frame by the chunk's start
            attitude:  v'_i = (2 S/m) (R(q_s) rho_i + eps_i e3) - g e3,  rho_i = 1/2 R(l_i) e3,  eps_i = 1/2 (1 - |l_i|^2).
This file restates that formulation in float64 numpy, step for step as the kernel orders it, and compares every
position, and the boundary states, with the sequential oracle: equality to rounding (1e-11), i.e. a reformulation, not
an approximation.  It also shows that the eps term is needed (without it the positions are off by far more than the
parity tolerance).  No GPU.
"""
from __future__ import annotations

import numpy as np
import pytest

from oracle import oracle as O
from paper_2509_14726_b200 import workloads as W


def qmul(a, b):
    return np.array([a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3],
                     a[0] * b[1] + a[1] * b[0] + a[2] * b[3] - a[3] * b[2],
                     a[0] * b[2] - a[1] * b[3] + a[2] * b[0] + a[3] * b[1],
                     a[0] * b[3] + a[1] * b[2] - a[2] * b[1] + a[3] * b[0]])


def rot(q):
    w, x, y, z = q
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                     [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                     [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])


def G(q, o):                       # q (x) (0, omega)
    return qmul(q, np.array([0.0, o[0], o[1], o[2]]))


def chunked_rollout(p, x0, T, L, with_eps=True):
    """positions after every step and (q, v, omega) at the chunk boundaries, the way the kernel computes them"""
    h, m, g = float(p["dt"]), float(p["mass"]), float(p["g"])
    lever = float(p["arm"]) / np.sqrt(2.0)
    ltx, lty, ltz = lever / float(p["Jx"]), lever / float(p["Jy"]), float(p["c_tau"]) / float(p["Jz"])
    gyx = (float(p["Jy"]) - float(p["Jz"])) / float(p["Jx"]); gyy = (float(p["Jz"]) - float(p["Jx"])) / float(p["Jy"])
    N = len(T)
    C = -(-N // L)
    s01, s23, d10, d23 = T[:, 0] + T[:, 1], T[:, 2] + T[:, 3], T[:, 1] - T[:, 0], T[:, 2] - T[:, 3]
    cm, ax, ay, az = (s01 + s23) / m, ltx * (s01 - s23), lty * (d10 + d23), ltz * (d23 - d10)
    chunks = [range(c * L, min((c + 1) * L, N)) for c in range(C)]

    def wstep(w, cx, z1, z2, z4):  # one RK4 step of w = omega_x + i omega_y (complex form of omega_xy_step)
        f = lambda w_, z: complex(gyx * w_.imag * z, gyy * z * w_.real) + cx
        k1 = f(w, z1); k2 = f(w + h / 2 * k1, z2); k3 = f(w + h / 2 * k2, z2); k4 = f(w + h * k3, z4)
        return w + h / 6 * (k1 + 2 * k2 + 2 * k3 + k4)

    # omega_z: prefix sums; omega_xy: affine maps of the chunks, composed in order
    oz_s = [x0[12] + h * az[:c * L].sum() for c in range(C)]
    maps = []
    for c, steps in enumerate(chunks):
        H, pp, oz = 1.0 + 0j, 0j, oz_s[c]
        for t in steps:
            z2, z4 = oz + h / 2 * az[t], oz + h * az[t]
            H = wstep(H, 0j, oz, z2, z4); pp = wstep(pp, complex(ax[t], ay[t]), oz, z2, z4)
            oz = oz + h * az[t]
        maps.append((H, pp))
    w_s, w = [], complex(x0[10], x0[11])
    for H, pp in maps:
        w_s.append(w); w = H * w + pp
    # chunk pass in the chunk's own frame
    l_end, V_end, Ve_end, P_loc, Pe_loc, om_end = [], [], [], [], [], []
    for c, steps in enumerate(chunks):
        o = np.array([w_s[c].real, w_s[c].imag, oz_s[c]])
        l = np.array(x0[3:7], float) if c == 0 else np.array([1.0, 0, 0, 0])
        V, Ve, Pr, Pe = np.zeros(3), 0.0, np.zeros(3), 0.0
        Pl, Pel = [], []
        for t in steps:
            a = np.array([ax[t], ay[t], az[t]])
            ko = lambda o_: np.array([gyx * o_[1] * o_[2] + a[0], gyy * o_[2] * o_[0] + a[1], a[2]])
            rho = lambda q_: np.array([q_[0] * q_[2] + q_[1] * q_[3], q_[2] * q_[3] - q_[0] * q_[1], 0.5 * (q_ @ q_) - (q_[1] ** 2 + q_[2] ** 2)])
            eps = lambda q_: 0.5 - 0.5 * (q_ @ q_) if with_eps else 0.0
            k1, g1 = ko(o), G(l, o); o2, l2 = o + h / 2 * k1, l + h / 4 * g1
            k2, g2 = ko(o2), G(l2, o2); o3, l3 = o + h / 2 * k2, l + h / 4 * g2
            k3, g3 = ko(o3), G(l3, o3); o4, l4 = o + h * k3, l + h / 2 * g3
            k4, g4 = ko(o4), G(l4, o4)
            r1, r2, r3, r4 = rho(l), rho(l2), rho(l3), rho(l4)
            e1, e2, e3, e4 = eps(l), eps(l2), eps(l3), eps(l4)
            kp, kv = cm[t] * h * h / 3, cm[t] * h / 3
            Pr = Pr + h * V + kp * (r1 + r2 + r3); Pe = Pe + h * Ve + kp * (e1 + e2 + e3) - h * h / 2 * g
            V = V + kv * (r1 + 2 * r2 + 2 * r3 + r4); Ve = Ve + kv * (e1 + 2 * e2 + 2 * e3 + e4) - h * g
            o = o + h / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
            n = l + h / 12 * (g1 + 2 * g2 + 2 * g3 + g4)
            l = n / np.linalg.norm(n)
            Pl.append(Pr.copy()); Pel.append(Pe)
        l_end.append(l); V_end.append(V); Ve_end.append(Ve); P_loc.append(Pl); Pe_loc.append(Pel); om_end.append(o)
    # join: attitudes (lane 0 carries q0), velocities, positions
    e3v = np.array([0.0, 0, 1.0])
    q_s, v_s, p_s = [np.array([1.0, 0, 0, 0])], [np.array(x0[7:10], float)], [np.array(x0[0:3], float)]
    acc = None
    pos, bq, bv, bo = [], [], [], []
    for c, steps in enumerate(chunks):
        R = rot(q_s[c])
        for j, t in enumerate(steps):
            pos.append(p_s[c] + (j + 1) * h * v_s[c] + R @ P_loc[c][j] + Pe_loc[c][j] * e3v)
        acc = l_end[c] if acc is None else qmul(acc, l_end[c])
        acc = acc / np.linalg.norm(acc)
        bq.append(acc.copy()); bo.append(om_end[c])
        v_next = v_s[c] + R @ V_end[c] + Ve_end[c] * e3v
        bv.append(v_next)
        q_s.append(acc.copy()); v_s.append(v_next); p_s.append(pos[-1])
    return np.array(pos), np.array(bq), np.array(bv), np.array(bo), [s[-1] for s in chunks]


def sequential(p, x0, T):
    xs, x = [], np.array(x0, float)
    for t in range(len(T)):
        x = O.rk4_step(p, x, T[t])
        xs.append(x.copy())
    return np.array(xs)


@pytest.mark.parametrize("N,L", [(50, 4), (64, 4), (20, 2), (7, 1), (33, 3)])
def test_chunked_formulation_equals_the_sequential_rk4(N, L):
    wl = W.cfg1()
    p = wl.params
    rng = np.random.default_rng(3)
    for case in range(4):
        x0 = wl.x0[0].astype(np.float64).copy()
        x0[10:13] = rng.normal(0, 4.0, 3)                   # spinning start: the affine-map scan matters
        x0[7:10] += rng.normal(0, 2.0, 3)
        q = rng.normal(0, 1, 4); x0[3:7] = q / np.linalg.norm(q) * (1.0 if case < 3 else 1.06)   # last case: |q0| != 1
        T = np.clip(float(p["mass"]) * float(p["g"]) / 4 + rng.normal(0, 1.5, (N, 4)), 0.0, 7.0)
        xs = sequential(p, x0, T)
        pos, bq, bv, bo, ends = chunked_rollout(p, x0, T, L)
        np.testing.assert_allclose(pos, xs[:, 0:3], rtol=0, atol=2e-11)
        np.testing.assert_allclose(bv, xs[ends, 7:10], rtol=0, atol=2e-11)
        np.testing.assert_allclose(bo, xs[ends, 10:13], rtol=0, atol=2e-10)
        np.testing.assert_allclose(bq, xs[ends, 3:7], rtol=0, atol=1e-12)


def test_the_eps_term_is_needed():
    # dropping eps_i = 1/2 (1 - |l_i|^2) treats the un-normalised stage quaternions as rotations: an error far above
    # the parity tolerance (1e-4 on costs of order 1 to 10), so the GPU parity tests do discriminate here
    wl = W.cfg1()
    p = wl.params
    rng = np.random.default_rng(5)
    x0 = wl.x0[0].astype(np.float64).copy()
    x0[10:13] = np.array([8.0, -6.0, 5.0])
    T = np.clip(float(p["mass"]) * float(p["g"]) / 4 + rng.normal(0, 1.5, (50, 4)), 0.0, 7.0)
    xs = sequential(p, x0, T)
    pos, *_ = chunked_rollout(p, x0, T, 4, with_eps=False)
    assert np.abs(pos - xs[:, 0:3]).max() > 1e-3
    pos, *_ = chunked_rollout(p, x0, T, 4, with_eps=True)
    assert np.abs(pos - xs[:, 0:3]).max() < 2e-11
