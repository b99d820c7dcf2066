"""Pins of the oracle's implementation of the paper's own contouring formulation (eq.(9) PAPER.md:149-161;
SURVEY.md NEXT-3): progress theta and its speed as states, the progress acceleration as a fifth sampled
input, path lookup by theta.  Readings R-33..R-37 of DESIGN.md."""
import numpy as np
import pytest

import definition_numpy as D
from oracle import oracle as O
from paper_2509_14726_b200 import workloads as W


def test_path_eval_on_a_square_and_a_circle():
    sq = np.array([[0, 0, 0], [2, 0, 0], [2, 2, 0], [0, 2, 0]], dtype=np.float64)      # closed, L = 8
    pos, tg, L = O.path_eval(sq, True, 1.0)
    assert L == pytest.approx(8.0)
    np.testing.assert_allclose(pos, [1, 0, 0], atol=1e-15)
    # vertex tangents are central differences: at (0,0) (1,-1)/sqrt2, at (2,0) (1,1)/sqrt2; mid-edge: (1,0)
    np.testing.assert_allclose(tg, [1, 0, 0], atol=1e-15)
    pos, tg, _ = O.path_eval(sq, True, 7.0)                   # on the closing segment (0,2) -> (0,0)
    np.testing.assert_allclose(pos, [0, 1, 0], atol=1e-15)
    np.testing.assert_allclose(tg, [0, -1, 0], atol=1e-15)
    for th in (9.0, -7.0, 17.0):                              # periodic in L
        np.testing.assert_allclose(O.path_eval(sq, True, th)[0], [1, 0, 0], atol=1e-12)
    np.testing.assert_allclose(O.path_eval(sq, True, 2.0)[0], [2, 0, 0], atol=1e-15)   # exactly a vertex
    # open path: clamped at both ends
    np.testing.assert_allclose(O.path_eval(sq, False, -3.0)[0], [0, 0, 0], atol=1e-15)
    np.testing.assert_allclose(O.path_eval(sq, False, 99.0)[0], [0, 2, 0], atol=1e-15)
    # a finely sampled circle: P(theta) and the tangent follow the analytic circle
    n, R = 720, 5.0
    a = np.linspace(0, 2 * np.pi, n, endpoint=False)
    circ = np.stack([R * np.cos(a), R * np.sin(a), np.zeros(n)], 1)
    for th in (0.3, 7.7, 20.0):
        pos, tg, L = O.path_eval(circ, True, th)
        ang = th / L * 2 * np.pi
        np.testing.assert_allclose(pos, [R * np.cos(ang), R * np.sin(ang), 0], atol=2e-4)
        np.testing.assert_allclose(tg, [-np.sin(ang), np.cos(ang), 0], atol=2e-4)
        assert np.linalg.norm(tg) == pytest.approx(1.0, abs=1e-15)


def test_progress_states_and_fifth_normal():
    P = dict(W.contour_paper(K=1, N=1).params)
    th, v = O.progress_step(P, 1.0, 2.0, 5.0)                  # constant acceleration over dt: exact
    h = float(P["dt"])
    assert th == pytest.approx(1.0 + h * 2.0 + 0.5 * h ** 2 * 5.0, abs=1e-15) and v == pytest.approx(2.0 + h * 5.0, abs=1e-15)
    assert O.progress_step(P, 0.0, 9.95, 20.0)[1] == pytest.approx(P["v_theta_max"])      # 10.35 -> 10
    assert O.progress_step(P, 0.0, 0.1, -20.0)[1] == 0.0                                  # -0.3 -> 0
    # the fifth normal is the first Box-Muller output of the Philox block at step t + 2^31
    assert O.normal5(3, 7, 11, 2, 1) == O.normals(3, 7, 11 + 2 ** 31, 2, 1)[0]
    assert O.normal5(3, 7, 11, 2, 1) not in O.normals(3, 7, 11, 2, 1)


def test_one_step_by_hand_on_a_straight_path():
    # path along +x through the origin; drone at (1, 0.3, 0.4) level at rest, theta = 0.6 (so P = (0.6,0,0)):
    # e = (0.4, 0.3, 0.4), e_l = 0.4, e_c^2 = 0.25.  K = 1, N = 1, sigma = sigma_v = 0 -> u = 0, dv = v_nom
    wl = W.contour_paper(K=1, N=1)
    p = dict(wl.params, sigma=0.0, sigma_v=0.0, w_limit=0.0, K=1, N=1)
    path = np.stack([np.linspace(-5, 5, 101), np.zeros(101), np.zeros(101)], 1)
    x0 = np.zeros((1, 19)); x0[0, 0:3] = (1.0, 0.3, 0.4); x0[0, 3] = 1.0
    x0[0, 13:17] = p["mass"] * p["g"] / 4; x0[0, 17] = 5.6; x0[0, 18] = 3.0     # s = x + 5 on this path
    r = O.step(p, O.Track(path=path, closed=False), x0, [0], np.zeros((1, 1, 4)), 0, 0, want_du=True,
               v_nom=np.array([[4.0]]))
    J = p["q_lag"] * 0.4 ** 2 + p["q_contour"] * 0.25 + p["r_dv"] * 16.0 - p["mu_progress"] * 3.0
    assert r["cost"][0, 0] == pytest.approx(J, rel=1e-12)
    np.testing.assert_allclose(r["v_new"], [[4.0]], atol=1e-15); np.testing.assert_allclose(r["dv"], 0.0, atol=1e-15)


def test_clamps_of_the_fifth_input_enter_the_update():
    wl = W.contour_paper(K=64, N=8)
    p = dict(wl.params, sigma_v=np.float32(60.0))
    r = O.step(p, O.Track(path=wl.path, closed=True), wl.x0, wl.start, wl.u_nom, 1, 0, want_du=True, v_nom=wl.v_nom)
    assert (np.abs(r["dv"]) == p["dv_max"]).mean() > 0.3 and np.abs(r["dv"]).max() <= p["dv_max"]
    np.testing.assert_allclose(r["v_new"][0], r["weights"][0] @ r["dv"][0], atol=1e-12)      # v_nom = 0
    k = int(np.argmin(r["cost"][0]))
    assert r["weights"][0, k] == r["weights"][0].max()


@pytest.mark.parametrize("kw,closed", [(dict(K=6, N=12), True), (dict(K=4, N=40), True), (dict(K=5, N=30), False)])
def test_brute_force_definition(kw, closed):
    wl = W.contour_paper(**kw)
    wl.v_nom = np.random.default_rng(3).uniform(-4, 4, wl.v_nom.shape).astype(np.float32)
    if not closed:                       # open form, theta_0 just before the end at the upper speed limit
        wl.closed = 0
        L = float(np.linalg.norm(np.diff(wl.path.astype(np.float64), axis=0), axis=1).sum())
        wl.x0[0, 17:19] = np.float32([L - 0.2, 10.0]); wl.x0[0, 0:3] = wl.path[-3]
    r = O.step(wl.params, O.Track(path=wl.path, closed=wl.closed), wl.x0, wl.start, wl.u_nom, 11, 3,
               want_du=True, v_nom=wl.v_nom)
    J, w, un, vn, du, dv = D.mppi_step5(wl.params, dict(path=wl.path.astype(np.float64), closed=wl.closed),
                                        wl.x0[0].astype(np.float64), wl.u_nom[0].astype(np.float64),
                                        wl.v_nom[0].astype(np.float64), 11, 3)
    np.testing.assert_allclose(r["cost"][0], J, rtol=1e-12, atol=1e-10)
    np.testing.assert_allclose(r["du"][0], du, rtol=0, atol=1e-13)
    np.testing.assert_allclose(r["dv"][0], dv, rtol=0, atol=1e-13)
    np.testing.assert_allclose(r["u_new"][0], un, rtol=0, atol=1e-12)
    np.testing.assert_allclose(r["v_new"][0], vn, rtol=0, atol=1e-12)


def test_plant_step_advances_the_progress_states_and_shifts_both_nominals():
    # [R-39] drone part = one rate-model RK4 step with u_new[0]; theta, v_theta by the closed form of a held
    # acceleration v_new[0]; both nominals shift by one with the last entry repeated
    wl = W.contour_paper(K=8, N=6)
    p = wl.params
    x0 = wl.x0.astype(np.float64); x0[0, 17:19] = (3.0, 9.9)
    u = np.linspace(-3, 3, 24).reshape(1, 6, 4)
    v = np.array([[7.0, -1.0, 2.0, 0.5, -4.0, 6.0]])
    x1, un, vn = O.sim_step_progress(p, x0, u, v)
    h = float(p["dt"])
    np.testing.assert_allclose(x1[0, :17], O.rk4_rate_step(p, x0[0, :17], u[0, 0]), atol=1e-15)
    assert x1[0, 17] == pytest.approx(3.0 + h * 9.9 + 0.5 * h * h * 7.0, abs=1e-15)
    assert x1[0, 18] == pytest.approx(min(9.9 + h * 7.0, float(p["v_theta_max"])), abs=1e-15) and x1[0, 18] == p["v_theta_max"]
    np.testing.assert_array_equal(un[0, :-1], u[0, 1:]); np.testing.assert_array_equal(un[0, -1], u[0, -1])
    np.testing.assert_array_equal(vn[0], [-1.0, 2.0, 0.5, -4.0, 6.0, 6.0])
    # hover + zero progress acceleration: the drone stays, theta advances uniformly
    x = wl.x0.astype(np.float64); x[0, 7:13] = 0.0; x[0, 17:19] = (1.0, 2.0)
    p0 = dict(p, drag_x=0.0, drag_y=0.0, drag_z=0.0)
    for _ in range(10):
        x, _, _ = O.sim_step_progress(p0, x, np.zeros((1, 6, 4)), np.zeros((1, 6)))
    np.testing.assert_allclose(x[0, :3], wl.x0[0, :3], atol=1e-7)
    assert x[0, 17] == pytest.approx(1.0 + 10 * h * 2.0, abs=1e-13) and x[0, 18] == 2.0
