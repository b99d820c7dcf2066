"""Pins of the oracle's implementation of the paper's own input model: control input
u = dT/dt with the four rotor thrusts as states, rate and thrust ranges of Table I
(PAPER.md:216-221), rotor drag of eq.(2) and the soft body-rate limit ("external cost",
PAPER.md:84).  Readings R-27..R-32 of DESIGN.md.  Closed forms, invariants, and the independently
written numpy evaluator."""
import numpy as np
import pytest

import definition_numpy as D
from oracle import oracle as O
from paper_2509_14726_b200 import workloads as W


def params(**over):
    p = W.base_params(input_model=1, rate_max=10.0, T_max=10.0, w_limit=1.0, omega_max=10.0)
    p.update(over)
    return p


def level(T, p=(0, 0, 0), v=(0, 0, 0), w=(0, 0, 0), q=(1, 0, 0, 0)):
    return np.array([*p, *q, *v, *w, *T], dtype=np.float64)


def test_hover_with_thrust_states_is_an_equilibrium():
    P = params(drag_x=0.25, drag_y=0.25, drag_z=0.1)
    hov = P["mass"] * P["g"] / 4
    x = level([hov] * 4, p=(1, 2, 3))
    for _ in range(20):
        x = O.rk4_rate_step(P, x, np.zeros(4))
    np.testing.assert_allclose(x, level([hov] * 4, p=(1, 2, 3)), rtol=0, atol=1e-13)


def test_equal_thrust_ramp_closed_form():
    # all four rates = a, level, no drag: T(t) = T0 + a t;  v_z' = 4 (T0 + a t)/m - g  ->  cubic p_z:
    # RK4 is exact for it
    P = params()
    a, T0, h = 3.0, P["mass"] * P["g"] / 4, P["dt"]
    x = level([T0] * 4)
    for k in range(1, 16):
        x = O.rk4_rate_step(P, x, np.full(4, a))
        t = k * h
        np.testing.assert_allclose(x[13:], T0 + a * t, rtol=0, atol=1e-13)
        assert x[9] == pytest.approx(4 * a / P["mass"] * t ** 2 / 2, abs=1e-13)
        assert x[2] == pytest.approx(4 * a / P["mass"] * t ** 3 / 6, abs=1e-13)
        np.testing.assert_allclose(x[3:7], [1, 0, 0, 0], atol=1e-15)
        np.testing.assert_allclose(x[10:13], 0, atol=1e-15)


def test_thrust_rate_differences_make_torque_with_the_right_sign():
    # rates (+a, +a, -a, -a): the thrust sum stays, tau_x = l/sqrt2 * 4 a t  ->  omega_x = 2 sqrt2 l a t^2 / Jx
    P = params()
    a, T0, h = 0.5, 2.0, P["dt"]
    x = level([T0] * 4)
    x = O.rk4_rate_step(P, x, np.array([a, a, -a, -a]))
    lever = P["arm"] / np.sqrt(2)
    assert x[10] == pytest.approx(lever * 4 * a * h ** 2 / 2 / P["Jx"], rel=1e-9)
    assert abs(x[11]) < 1e-12 and abs(x[12]) < 1e-12
    np.testing.assert_allclose(x[13:], [T0 + a * h, T0 + a * h, T0 - a * h, T0 - a * h], atol=1e-15)


def test_thrust_states_are_projected_onto_their_range():
    P = params()
    x = O.rk4_rate_step(P, level([9.95, 0.05, 5.0, 5.0]), np.array([10.0, -10.0, 0.0, 0.0]))
    np.testing.assert_allclose(x[13:], [10.0, 0.0, 5.0, 5.0], atol=1e-15)       # 10.15 -> 10, -0.15 -> 0


def test_drag_decay_is_the_rk4_polynomial_and_follows_the_attitude():
    # level hover, velocity along world x = body x:  v_x' = -d_x v_x.  One RK4 step multiplies by the
    # degree-4 Taylor polynomial of exp(-d h); over many steps it follows exp(-d t)
    P = params(drag_x=0.4, drag_y=0.9, drag_z=0.2)
    hov = P["mass"] * P["g"] / 4
    z = P["drag_x"] * P["dt"]
    x = O.rk4_rate_step(P, level([hov] * 4, v=(2, 0, 0)), np.zeros(4))
    assert x[7] == pytest.approx(2 * (1 - z + z ** 2 / 2 - z ** 3 / 6 + z ** 4 / 24), rel=1e-14)
    assert abs(x[8]) < 1e-15 and abs(x[9]) < 1e-13
    x = level([hov] * 4, v=(2, 0, 0))
    for _ in range(100):
        x = O.rk4_rate_step(P, x, np.zeros(4))
    assert x[7] == pytest.approx(2 * np.exp(-P["drag_x"] * 100 * P["dt"]), rel=1e-9)
    # yawed by 90 degrees the body y axis points along world -x... the world-x velocity now feels d_y
    q = (np.cos(np.pi / 4), 0, 0, np.sin(np.pi / 4))
    x = O.rk4_rate_step(P, level([hov] * 4, v=(2, 0, 0), q=q), np.zeros(4))
    zy = P["drag_y"] * P["dt"]
    assert x[7] == pytest.approx(2 * (1 - zy + zy ** 2 / 2 - zy ** 3 / 6 + zy ** 4 / 24), rel=1e-12)
    # the same drag acts in the 13-state thrust-input model through the shared f_dyn
    P0 = dict(P, input_model=0)
    y = O.rk4_step(P0, level([hov] * 4, v=(2, 0, 0))[:13], np.full(4, hov))
    assert y[7] == pytest.approx(2 * (1 - z + z ** 2 / 2 - z ** 3 / 6 + z ** 4 / 24), rel=1e-14)


def test_body_rate_limit_cost():
    P = params(w_limit=0.5, omega_max=10.0)
    assert O.rate_limit_cost(P, (12.0, -11.0, 5.0)) == pytest.approx(0.5 * (4.0 + 1.0), abs=1e-15)
    assert O.rate_limit_cost(P, (10.0, -10.0, 0.0)) == 0.0


def test_rollout_clamps_rates_and_costs_the_limit_and_the_rates():
    # K=1, N=1 by hand: u = clamp(u_nom + sigma z, -rate_max, rate_max); tracking: J = state term at x0
    # + R |u|^2 + terminal state term, + limit cost of the post-step rates
    wl = W.rate_track(K=1, N=1)
    p = dict(wl.params, sigma=np.float32(40.0), w_limit=np.float32(2.0), omega_max=np.float32(0.01))
    trk = O.Track(ref=wl.ref)
    r = O.step(p, trk, wl.x0, wl.start, wl.u_nom, 0, 0, want_du=True)
    z = O.normals(0, 0, 0, 0, 0)
    u = np.clip(p["sigma"] * z, -p["rate_max"], p["rate_max"])
    assert (np.abs(u) == p["rate_max"]).any()                    # the clamp acts
    np.testing.assert_allclose(r["du"][0, 0, 0], u, atol=1e-15)
    x1 = O.rk4_rate_step(p, wl.x0[0], u)
    ref = wl.ref.astype(np.float64)
    J = (O.track_state_term(p, wl.x0[0, :13], ref[0]) + p["R"] * np.sum(u ** 2)
         + O.track_state_term(p, x1[:13], ref[1]) + O.rate_limit_cost(p, x1[10:13]))
    assert r["cost"][0, 0] == pytest.approx(J, rel=1e-13)
    assert O.rate_limit_cost(p, x1[10:13]) > 0
    np.testing.assert_allclose(r["u_new"][0, 0], u, atol=1e-15)   # K = 1: the sample itself


def _dict_track(wl):
    f = lambda a: None if a is None else a.astype(np.float64)
    return dict(gates=f(wl.gates), ref=f(wl.ref), path=f(wl.path), closed=wl.closed, prev_front=wl.prev_front)


@pytest.mark.parametrize("name,kw", [("rate_gate_paper", dict(K=6, N=12)), ("rate_track", dict(K=6, N=5)),
                                     ("rate_stress", dict(K=12, N=30))])
def test_brute_force_definition(name, kw):
    wl = W.ALL[name](**kw)
    trk = O.Track(gates=wl.gates, ref=wl.ref, path=wl.path, closed=wl.closed, prev_front=wl.prev_front)
    r = O.step(wl.params, trk, wl.x0, wl.start, wl.u_nom, 11, 3, want_du=True)
    J, w, un, du = D.mppi_step(wl.params, _dict_track(wl), wl.x0[0].astype(np.float64), int(wl.start[0]),
                               wl.u_nom[0].astype(np.float64), 11, 3)
    np.testing.assert_allclose(r["cost"][0], J, rtol=1e-12, atol=1e-10)
    np.testing.assert_allclose(r["du"][0], du, rtol=0, atol=1e-13)
    np.testing.assert_allclose(r["weights"][0], w, rtol=1e-9, atol=1e-15)
    np.testing.assert_allclose(r["u_new"][0], un, rtol=0, atol=1e-12)


def test_stress_case_saturates_thrusts_and_crosses_gates():
    wl = W.rate_stress(K=256, N=30)
    r = O.step(wl.params, O.Track(gates=wl.gates), wl.x0, wl.start, wl.u_nom, wl.seed, 0, want_du=True)
    assert (r["ncross"][0] > 0).sum() >= 20 and (r["ncross"][0] == 0).sum() >= 20
    assert (np.abs(r["du"]) == wl.params["rate_max"]).mean() > 0.05      # rate clamp acts at scale


def test_plant_step_and_front_flags_under_the_rate_model():
    # plant: one rate-model RK4 step with u_new[0], thrust states advance, nominal shifts [R-14]
    wl = W.rate_gate_paper(K=8, N=6)
    p = wl.params
    trk = O.Track(gates=wl.gates)
    u = np.linspace(-3, 3, 24).reshape(1, 6, 4)
    x1, s1, un = O.sim_step(p, trk, wl.x0, wl.start, u)
    np.testing.assert_allclose(x1[0], O.rk4_rate_step(p, wl.x0[0], u[0, 0]), atol=1e-15)
    np.testing.assert_allclose(x1[0, 13:], wl.x0[0, 13:].astype(np.float64) + p["dt"] * u[0, 0], atol=1e-15)
    np.testing.assert_array_equal(un[0, :-1], u[0, 1:]); np.testing.assert_array_equal(un[0, -1], u[0, -1])
    # flags: free fall under the rate model (T = 0, u = 0) against the closed form, as in the thrust model
    pf = dict(W.base_params(N=40, objective=W.OBJ_GATE_PAPER), input_model=1, rate_max=10.0, T_max=10.0)
    g = np.array([[0, 0, 1.0, 0, 0, -1, 1, 0, 0, 5, 5]], dtype=np.float64)
    x0 = np.zeros(17); x0[2] = 2.0; x0[3] = 1.0
    f, _ = O.front_flags(pf, O.Track(gates=g), x0, 0, np.zeros((40, 4)))
    k = np.arange(41)
    np.testing.assert_array_equal(f, (k * pf["dt"] < np.sqrt(2 * 1.0 / pf["g"])).astype(np.int32))
