"""Pins P9, P11, P14 and the worked example: one full MPPI iteration of the
oracle (Alg. 1; weights eq.(4), update eq.(5)) against hand results, softmax
invariants and the independently written numpy evaluator in tests/definition_numpy.py."""
import numpy as np
import pytest

import definition_numpy as D
from oracle import oracle as O
from paper_2509_14726_b200 import workloads as W


def _golden(golden_dir):
    vals = {}
    for line in (golden_dir / "worked_example_cfg0.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        vals[k] = np.array([float(t) for t in v])
    return vals


def exact_cfg0_params(**over):
    # the worked example uses the decimal constants of BASELINE.json configs[0] exactly
    p = dict(K=1, N=1, B=1, objective=0, dt=0.02, sigma=1.0, mass=0.85, Jx=1e-3, Jy=1e-3,
             Jz=1.7e-3, arm=0.15, c_tau=0.016, g=9.81, T_min=0.0, T_max=7.0, w_omega=0.01,
             gate_miss_penalty=10.0, gate_pass_bonus=5.0, Qp=100.0, Qv=1.0, Qq=10.0, Qw=0.1,
             R=0.01, q_contour=200.0, q_lag=50.0, mu_progress=2.0, window=16)
    p["lambda"] = 1.0
    p.update(over)
    return p


def test_worked_example_one_sample_step(golden_dir):
    g = _golden(golden_dir)
    p = exact_cfg0_params()
    gates = np.array([[5, 0, 1.5, 0, 1, 0, 1, 0, 0, .75, .75], [0, 5, 1.5, -1, 0, 0, 0, 1, 0, .75, .75],
                      [-5, 0, 1.5, 0, -1, 0, -1, 0, 0, .75, .75], [0, -5, 1.5, 1, 0, 0, 0, -1, 0, .75, .75]],
                     dtype=float)
    x0 = np.array([[5, -2, 1.5, 1, 0, 0, 0, 0, 0, 0, 0, 0, 0]], dtype=float)
    hover = 0.85 * 9.81 / 4
    assert hover == pytest.approx(g["hover"][0], abs=1e-12)
    u_nom = np.full((1, 1, 4), hover)
    r = O.step(p, O.Track(gates=gates), x0, [0], u_nom, 0, 0, want_du=True)
    T = u_nom[0, 0] + r["du"][0, 0, 0]
    np.testing.assert_allclose(T, g["T"], atol=2e-12)
    x1 = O.rk4_step(p, x0[0], T)
    np.testing.assert_allclose(x1[0:3], g["p1"], atol=2e-12)
    np.testing.assert_allclose(x1[3:7], g["q1"], atol=2e-9)      # q1[1] is printed to 9 digits
    np.testing.assert_allclose(x1[7:10], g["v1"], atol=2e-12)
    np.testing.assert_allclose(x1[10:13], g["w1"], atol=2e-12)
    assert np.linalg.norm(x1[0:3] - gates[0, 0:3]) == pytest.approx(g["d1"][0], abs=2e-12)
    assert r["cost"][0, 0] == pytest.approx(g["J"][0], abs=2e-12)
    # K = 1: the only sample takes all the weight and u_new is that sample (P9)
    assert r["weights"][0, 0] == 1.0
    np.testing.assert_allclose(r["u_new"][0, 0], T, atol=1e-15)
    # hand check of omega: tau / J * dt up to the gyroscopic coupling
    lever = 0.15 / np.sqrt(2)
    tau = np.array([lever * (T[0] + T[1] - T[2] - T[3]) / 1e-3, lever * (-T[0] + T[1] + T[2] - T[3]) / 1e-3,
                    0.016 * (T[0] - T[1] + T[2] - T[3]) / 1.7e-3]) * 0.02
    np.testing.assert_allclose(x1[10:13], tau, atol=0.01)


def test_k1_n1_sigma0_by_hand():
    # P9: sigma = 0, equal thrusts: v_z = (S/m - g) dt, p_z = (S/m - g) dt^2 / 2, cost = d1 - d0
    p = exact_cfg0_params(sigma=0.0)
    gates = np.array([[5, 0, 1.5, 0, 1, 0, 1, 0, 0, .75, .75]] * 2, dtype=float)
    x0 = np.array([[5, -2, 1.5, 1, 0, 0, 0, 0, 0, 0, 0, 0, 0]], dtype=float)
    u = np.full((1, 1, 4), 3.0)
    r = O.step(p, O.Track(gates=gates), x0, [0], u, 0, 0, want_du=True)
    a = 12.0 / 0.85 - 9.81
    d1 = np.hypot(2.0, 0.5 * a * 0.02 ** 2)
    assert r["cost"][0, 0] == pytest.approx(d1 - 2.0, abs=1e-14)
    assert np.all(r["du"] == 0) and np.all(r["u_new"] == 3.0) and r["weights"][0, 0] == 1.0


def test_clamp_enters_the_update():
    # [R-8]: du is the clamped perturbation; with a nominal at the upper limit du <= 0 everywhere
    p = exact_cfg0_params(K=64, N=4, sigma=2.0)
    gates = np.array([[5, 0, 1.5, 0, 1, 0, 1, 0, 0, .75, .75]] * 2, dtype=float)
    x0 = np.array([[5, -2, 1.5, 1, 0, 0, 0, 0, 0, 0, 0, 0, 0]], dtype=float)
    u = np.full((1, 4, 4), 7.0)
    r = O.step(p, O.Track(gates=gates), x0, [0], u, 1, 0, want_du=True)
    assert r["du"].max() == 0.0 and r["du"].min() >= -7.0 and (r["du"] == 0).mean() > 0.4
    assert r["u_new"].max() <= 7.0 and r["u_new"].min() >= 0.0
    for k in (0, 5):
        z = O.normals(1, k, 2, 0, 0)
        np.testing.assert_allclose(r["du"][0, k, 2], np.clip(7.0 + 2.0 * z, 0, 7) - 7.0, atol=1e-15)


# ---- P11: softmax / update invariants -------------------------------------------------------

def test_weights_invariants():
    rng = np.random.default_rng(0)
    K, N = 200, 7
    cost = rng.normal(size=K) * 5 + 100
    du = rng.normal(size=(K, N, 4)); u = rng.normal(size=(N, 4))
    w, un = O.weights_update(0.7, cost, du, u)
    assert abs(w.sum() - 1) < 1e-12 and w.min() >= 0
    e = np.exp(-cost / 0.7)
    np.testing.assert_allclose(w, e / e.sum(), rtol=1e-10)            # eq.(4) literally
    np.testing.assert_allclose(un, u + np.tensordot(w, du, axes=(0, 0)), atol=1e-13)   # eq.(5)
    w2, un2 = O.weights_update(0.7, cost + 1234.5, du, u)               # shift invariance
    np.testing.assert_allclose(w2, w, rtol=1e-9); np.testing.assert_allclose(un2, un, atol=1e-11)
    # huge costs do not overflow
    w3, _ = O.weights_update(0.5, cost * 1e4, du, u)
    assert np.isfinite(w3).all() and abs(w3.sum() - 1) < 1e-12


def test_weights_equal_costs_and_lambda_to_zero():
    rng = np.random.default_rng(1)
    du = rng.normal(size=(2, 3, 4)); u = rng.normal(size=(3, 4))
    w, un = O.weights_update(1.0, [4.0, 4.0], du, u)
    np.testing.assert_allclose(w, [0.5, 0.5]); np.testing.assert_allclose(un, u + du.mean(0), atol=1e-15)
    K = 50
    cost = rng.normal(size=K); du = rng.normal(size=(K, 3, 4))
    w, un = O.weights_update(1e-6, cost, du, u)
    k = int(np.argmin(cost))
    assert w[k] == 1.0 and w.sum() == 1.0
    np.testing.assert_allclose(un, u + du[k], atol=1e-15)
    # larger lambda flattens, smaller sharpens
    wa, _ = O.weights_update(10.0, cost, du, u); wb, _ = O.weights_update(0.1, cost, du, u)
    assert wb.max() > wa.max()


def test_update_is_inside_the_sample_hull():
    wl = W.cfg0(K=64, N=10)
    r = O.step(wl.params, O.Track(gates=wl.gates), wl.x0, wl.start, wl.u_nom, 0, 0, want_du=True)
    s = wl.u_nom[0].astype(np.float64) + r["du"][0]
    assert (r["u_new"][0] <= s.max(0) + 1e-12).all() and (r["u_new"][0] >= s.min(0) - 1e-12).all()
    w, un = O.weights_update(wl.params["lambda"], r["cost"][0], r["du"][0], wl.u_nom[0])
    np.testing.assert_array_equal(w, r["weights"][0]); np.testing.assert_array_equal(un, r["u_new"][0])


# ---- P14: independent brute force, all three objectives ------------------------------------

def _as_dict_track(wl):
    return dict(gates=None if wl.gates is None else wl.gates.astype(np.float64),
                ref=None if wl.ref is None else wl.ref.astype(np.float64),
                path=None if wl.path is None else wl.path.astype(np.float64), closed=wl.closed)


@pytest.mark.parametrize("name,kw", [("cfg0", dict(K=8, N=3)), ("stress_gate", dict(K=8, N=30)),
                                     ("cfg2", dict(K=8, N=3)), ("cfg3", dict(K=8, N=3)),
                                     ("cfg1", dict(K=4, N=25)), ("cfg2", dict(K=4, N=25)),
                                     ("cfg3", dict(K=4, N=25))])
def test_brute_force_definition(name, kw):
    wl = W.ALL[name](**kw)
    trk = O.Track(gates=wl.gates, ref=wl.ref, path=wl.path, closed=wl.closed)
    it = 3
    r = O.step(wl.params, trk, wl.x0, wl.start, wl.u_nom, 11, it, want_du=True)
    J, w, un, du = D.mppi_step(wl.params, _as_dict_track(wl), wl.x0[0].astype(np.float64),
                               int(wl.start[0]), wl.u_nom[0].astype(np.float64), 11, it)
    np.testing.assert_allclose(r["cost"][0], J, rtol=1e-12, atol=1e-12)
    np.testing.assert_allclose(r["du"][0], du, rtol=0, atol=1e-14)
    np.testing.assert_allclose(r["weights"][0], w, rtol=1e-9, atol=1e-15)
    np.testing.assert_allclose(r["u_new"][0], un, rtol=0, atol=1e-12)


def test_brute_force_sees_gate_events():
    # the stress case must really exercise pass and miss branches in both implementations
    wl = W.stress_gate(K=64, N=30)
    r = O.step(wl.params, O.Track(gates=wl.gates), wl.x0, wl.start, wl.u_nom, wl.seed, 0)
    assert (r["ncross"] > 0).sum() >= 10 and (r["ncross"] == 0).sum() >= 5
    trk = _as_dict_track(wl)
    for k in (0, 1, 2, 3, 10, 33):
        J, _, aux = D.rollout_cost(wl.params, trk, wl.x0[0].astype(np.float64), 0,
                                   wl.u_nom[0].astype(np.float64), wl.seed, 0, k, 0)
        assert r["cost"][0, k] == pytest.approx(J, rel=1e-12, abs=1e-12)
        assert r["aux_end"][0, k] == aux


def test_controller_index_feeds_the_counter():
    # B = 2 identical controllers get independent noise (counter word 3 = b) [R-18]
    wl = W.cfg0(K=16, N=4)
    p = dict(wl.params); p["B"] = 2
    x0 = np.repeat(wl.x0, 2, 0); u = np.repeat(wl.u_nom, 2, 0)
    r = O.step(p, O.Track(gates=wl.gates), x0, [0, 0], u, 0, 0, want_du=True)
    assert not np.allclose(r["du"][0], r["du"][1])
    np.testing.assert_allclose(r["du"][1, 3, 2], np.clip(u[1, 2] + p["sigma"] * O.normals(0, 3, 2, 0, 1),
                                                         0, 7) - u[1, 2], atol=1e-15)


def test_sim_step_gate_shift_and_advance():
    wl = W.stress_gate(K=32, N=6)
    p = wl.params
    trk = O.Track(gates=wl.gates)
    u_new = np.arange(24, dtype=np.float64).reshape(1, 6, 4) * 0.1 + 1.0
    x = wl.x0.astype(np.float64)
    start = np.array([0], np.int32)
    passed = False
    x[0, 7:10] *= 2.0                          # 12 m/s from 3 m before the gate: crosses in ~13 steps
    for _ in range(20):
        xn, start_n, nxt = O.sim_step(p, trk, x, start, u_new)
        np.testing.assert_allclose(xn[0], O.rk4_step(p, x[0], u_new[0, 0]), atol=0)
        np.testing.assert_array_equal(nxt[0, :-1], u_new[0, 1:]); np.testing.assert_array_equal(nxt[0, -1], u_new[0, -1])
        if start_n[0] != start[0]:
            passed = True
            c, n = wl.gates[0, 0:3], wl.gates[0, 3:6]
            assert n @ (x[0, 0:3] - c) < 0 <= n @ (xn[0, 0:3] - c)
        x, start = xn, start_n
    assert passed and start[0] == 1


def test_brute_force_contour_wraps_the_closed_path():
    # start just before the seam of the periodic path, flying along it at 8 m/s: the arc-length
    # progress must be wrapped into (-L/2, L/2] when the nearest index jumps from P-1 to 0
    wl = W.cfg3(K=4, N=25)
    pts = wl.path.astype(np.float64)
    tan = pts[496] - pts[494]; tan /= np.linalg.norm(tan)
    x0 = np.zeros(13); x0[0:3] = pts[495] + [0.1, 0.05, -0.1]; x0[3] = 1; x0[7:10] = 8 * tan
    x0 = x0.astype(np.float32)[None]
    trk = O.Track(path=wl.path, closed=True)
    r = O.step(wl.params, trk, x0, [-1], wl.u_nom, 2, 0)
    assert r["aux_end"][0].min() < 200           # index wrapped past the seam
    J, w, un, du = D.mppi_step(wl.params, _as_dict_track(wl), x0[0].astype(np.float64), -1,
                               wl.u_nom[0].astype(np.float64), 2, 0)
    np.testing.assert_allclose(r["cost"][0], J, rtol=1e-12)
    # the progress reward really is positive: cost with mu = 0 is larger
    p0 = dict(wl.params); p0["mu_progress"] = 0.0
    r0 = O.step(p0, trk, x0, [-1], wl.u_nom, 2, 0)
    d = (r0["cost"][0] - r["cost"][0]) / wl.params["mu_progress"]
    assert (d > 2.0).all() and (d < 6.0).all()     # ~4 m flown in 0.5 s


# ---- closed-loop glue under tracking and contouring (Alg. 1 l.2-3 PAPER.md:177-178; receding horizon
# PAPER.md:57, 97; oracle/mppi_oracle.c orc_sim_step).  The plant input is zero thrust, so the new position
# is the free-fall closed form p + v dt - g dt^2/2 e_z (pinned by P4) and every expected index below is
# worked out by hand from it.

def _free_fall_params(**over):
    return exact_cfg0_params(**dict(dict(K=32, N=4, T_min=0.0), **over))


def test_sim_step_tracking_clock_advances_and_clamps_at_the_margin():
    # reference with a 3-row margin: M = N + 1 + 3 rows -> the start row may be 0..3 (= M - 1 - N);
    # start -> start + 1 per control step, then stays clamped; the rows' content plays no role
    N = 4
    p = _free_fall_params(objective=1, N=N)
    M = N + 1 + 3
    ref = np.zeros((M, 13)); ref[:, 3] = 1.0
    trk = O.Track(ref=ref)
    x = np.zeros((1, 13)); x[0, 0:3] = (1.0, 2.0, 30.0); x[0, 3] = 1.0; x[0, 7:10] = (3.0, -1.0, 0.5)
    u_new = np.zeros((1, N, 4)); u_new[0, :, 0] = np.arange(N) + 1.0      # thrust 1 N on rotor 0 at step 0 only matters
    u_new[0, 0] = 0.0                                                     # the plant applies u_new[0] = 0: free fall
    start = np.array([0], np.int32)
    seen = []
    for step in range(6):
        xn, start_n, nxt = O.sim_step(p, trk, x, start, u_new)
        t = p["dt"]
        np.testing.assert_allclose(xn[0, 0:3], x[0, 0:3] + x[0, 7:10] * t - [0, 0, 0.5 * p["g"] * t * t], atol=1e-13)
        np.testing.assert_array_equal(nxt[0, :-1], u_new[0, 1:]); np.testing.assert_array_equal(nxt[0, -1], u_new[0, -1])
        seen.append(int(start_n[0]))
        x, start = xn, start_n
    assert seen == [1, 2, 3, 3, 3, 3]                     # M - 1 - N = 3
    # a start row beyond the margin is pulled back to it, a row far below it still advances by one
    _, s2, _ = O.sim_step(p, trk, x, np.array([17], np.int32), u_new)
    assert s2[0] == 3
    # with no margin at all (M = N + 1) the clock cannot move
    trk0 = O.Track(ref=ref[:N + 1])
    _, s3, _ = O.sim_step(p, trk0, x, np.array([0], np.int32), u_new)
    assert s3[0] == 0


def test_sim_step_contour_windowed_global_tie_and_seam():
    # straight OPEN path along x, vertices at 0.125 i (binary-exact), i = 0..39, window 3
    N = 4
    p = _free_fall_params(objective=2, N=N, window=3)
    pts = np.zeros((40, 3)); pts[:, 0] = 0.125 * np.arange(40); pts[:, 2] = 1.0
    trk = O.Track(path=pts, closed=False)
    u_new = np.zeros((1, N, 4))
    dt = p["dt"]

    def plant_at(px, vx=0.0):
        x = np.zeros((1, 13)); x[0, 0:3] = (px, 0.25, 1.0); x[0, 3] = 1.0; x[0, 7] = vx
        return x
    # the plant moves 5 m/s * 0.02 s = 0.1 m: from x = 2.53 to 2.63 -> global nearest vertex 21 (2.625)
    x = plant_at(2.53, 5.0)
    xn, s, _ = O.sim_step(p, trk, x, np.array([-1], np.int32), u_new)
    assert xn[0, 0] == pytest.approx(2.53 + 5.0 * dt, abs=1e-14) and s[0] == 21
    # windowed around the hint 17 (vertices 14..20): the nearest INSIDE the window is 20, not 21
    _, s, _ = O.sim_step(p, trk, x, np.array([17], np.int32), u_new)
    assert s[0] == 20
    # hint 21 +- 3 contains the global minimiser
    _, s, _ = O.sim_step(p, trk, x, np.array([21], np.int32), u_new)
    assert s[0] == 21
    # the NEW position decides, not the old one: from 2.53 the old nearest vertex is 20 (2.5)
    assert np.argmin(np.abs(pts[:, 0] - 2.53)) == 20
    # exact tie between vertices 20 and 21 (x = 2.5625, no horizontal motion): first in scan order wins,
    # globally (ascending index) and in a window
    x = plant_at(2.5625, 0.0)
    for hint in (-1, 22, 19):
        _, s, _ = O.sim_step(p, trk, x, np.array([hint], np.int32), u_new)
        assert s[0] == 20
    # open path: a window hanging over the end is cut, never wrapped
    x = plant_at(0.01, 0.0)
    _, s, _ = O.sim_step(p, trk, x, np.array([38], np.int32), u_new)
    assert s[0] == 35                                        # window 35..39 (41 cut off): its nearest is 35
    # CLOSED path: 16 vertices on a circle of radius 2; hint 15, window 3 -> scan 12,13,14,15,0,1,2
    a = 2 * np.pi * np.arange(16) / 16
    circ = np.stack([2 * np.cos(a), 2 * np.sin(a), np.ones(16)], 1)
    trkc = O.Track(path=circ, closed=True)
    x = np.zeros((1, 13)); x[0, 0:3] = circ[1] * 1.1; x[0, 3] = 1.0       # next to vertex 1, across the seam from the hint
    _, s, _ = O.sim_step(p, trkc, x, np.array([15], np.int32), u_new)
    assert s[0] == 1
    # the same hint on the open form of the circle cannot reach vertex 1: window 12..15
    trko = O.Track(path=circ, closed=False)
    _, s, _ = O.sim_step(p, trko, x, np.array([15], np.int32), u_new)
    assert s[0] == 15
    # tie across the seam on a square ring with binary-exact vertices (0.5 m apart, 16 of them): the point
    # (-0.25, 0.25) is exactly as far from vertex 15 = (0, 0.5) as from vertex 0 = (0, 0).  The windowed scan
    # runs in offset order (12..15, then 0..2) and meets 15 first, although 0 is the smaller index; the
    # global scan (0..15) returns 0  [R-12]
    sq = np.array([(0, 0), (.5, 0), (1, 0), (1.5, 0), (2, 0), (2, .5), (2, 1), (2, 1.5), (2, 2), (1.5, 2), (1, 2), (.5, 2),
                   (0, 2), (0, 1.5), (0, 1), (0, .5)], float)
    sq = np.concatenate([sq, np.ones((16, 1))], 1)
    trks = O.Track(path=sq, closed=True)
    x[0, 0:3] = (-0.25, 0.25, 1.0); x[0, 7:10] = 0.0
    _, s, _ = O.sim_step(p, trks, x, np.array([15], np.int32), u_new)
    assert s[0] == 15
    _, s, _ = O.sim_step(p, trks, x, np.array([1], np.int32), u_new)       # scan 14, 15, 0, 1, ...: still 15 first
    assert s[0] == 15
    _, s, _ = O.sim_step(p, trks, x, np.array([-1], np.int32), u_new)
    assert s[0] == 0


def test_start_index_is_clamped_or_wrapped_as_the_interface_states():
    # include/mppi.h, mppi_step: tracking -- "reference row t0 ... clamped so that t0+N <= M-1"; gate objectives --
    # "index of the current target gate (wrapped mod G)" [R-10],[R-11]
    wl = W.cfg2(K=32, N=6, extra_rows=3)                      # M = N + 1 + 3: rows 0..3 are valid starts
    trk = O.Track(ref=wl.ref)
    J = lambda s: O.step(wl.params, trk, wl.x0, [s], wl.u_nom, 1, 0)["cost"]
    np.testing.assert_array_equal(J(7), J(3)); np.testing.assert_array_equal(J(4), J(3))
    np.testing.assert_array_equal(J(-2), J(0))
    assert not np.array_equal(J(2), J(3))
    # the clamped start really uses rows 3..9: the terminal row is the reference's last one
    x_end = wl.ref[3 + 6].astype(np.float64)
    p0 = dict(wl.params, K=32, sigma=0.0, Qv=0.0, Qq=0.0, Qw=0.0, R=0.0, Qp=1.0)
    x0 = np.tile(x_end, (1, 1)); x0[0, 7:13] = 0.0; x0[0, 3:7] = (1, 0, 0, 0)
    r = O.step(p0, trk, x0, [99], wl.u_nom, 1, 0)
    xs = [x0[0]]
    for t in range(6):
        xs.append(O.rk4_step(p0, xs[-1], wl.u_nom[0, t]))
    want = sum(np.sum((xs[t][0:3] - wl.ref[3 + t, 0:3].astype(np.float64)) ** 2) for t in range(7))
    assert r["cost"][0, 0] == pytest.approx(want, rel=1e-12)
    wl = W.stress_gate(K=32, N=10)
    trk = O.Track(gates=wl.gates)
    G = wl.gates.shape[0]
    Jg = lambda s: O.step(wl.params, trk, wl.x0, [s], wl.u_nom, 1, 0)["cost"]
    np.testing.assert_array_equal(Jg(G + 1), Jg(1)); np.testing.assert_array_equal(Jg(-1), Jg(G - 1))
    assert not np.array_equal(Jg(0), Jg(1))


def test_unrepresentable_costs_are_capped_and_get_no_weight():
    # [R-41] (include/mppi.h conventions): a rollout whose cost is NaN or beyond the fp32 range counts as 3.0e38.
    # A miss penalty of 3e38 pushes every sample that misses the gate over the cap; the samples that pass keep their
    # costs and share the whole weight
    wl = W.stress_gate(K=256, N=30)
    p = dict(wl.params, gate_miss_penalty=3.0e38)
    trk = O.Track(gates=wl.gates)
    r = O.step(p, trk, wl.x0, wl.start, wl.u_nom, wl.seed, 0, want_du=True)
    r0 = O.step(wl.params, trk, wl.x0, wl.start, wl.u_nom, wl.seed, 0)
    J, J0 = r["cost"][0], r0["cost"][0]
    missed = np.abs(J - J0) > 1.0                                  # the samples whose cost holds a miss penalty
    assert missed.sum() >= 20 and (~missed).sum() >= 20
    assert (J[missed] == 3.0e38).all() and np.isfinite(J).all()
    np.testing.assert_array_equal(J[~missed], J0[~missed])
    w = r["weights"][0]
    assert (w[missed] == 0.0).all() and w.sum() == pytest.approx(1.0, abs=1e-12)
    z = np.exp(-(J[~missed] - J[~missed].min()) / p["lambda"])
    np.testing.assert_allclose(w[~missed], z / z.sum(), rtol=1e-12)
    # every sample over the cap: all weigh the same, the update is the plain mean of the clamped samples
    wl2 = W.cfg2(K=32, N=4)
    p2 = dict(wl2.params, Qp=3.0e38)
    x0 = wl2.x0.copy(); x0[0, 0] += 10.0
    r2 = O.step(p2, O.Track(ref=wl2.ref), x0, wl2.start, wl2.u_nom, 1, 0, want_du=True)
    assert (r2["cost"] == 3.0e38).all()
    np.testing.assert_allclose(r2["weights"], 1.0 / 32, rtol=1e-12)
    np.testing.assert_allclose(r2["u_new"][0], wl2.u_nom[0] + r2["du"][0].mean(0), atol=1e-12)
