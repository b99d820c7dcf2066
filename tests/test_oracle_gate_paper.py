"""Pins of the oracle's implementation of the paper's own gate-progress objective (eq.(6),(7) and the
temporal gate-switching check of Fig. 2; readings R-23..R-26 of DESIGN.md):
hand-built single segments, closed forms, and the independently written numpy evaluator."""
import numpy as np
import pytest

import definition_numpy as D
from oracle import oracle as O
from paper_2509_14726_b200 import workloads as W


@pytest.fixture()
def P():
    return W.base_params(objective=W.OBJ_GATE_PAPER, q_near=2.0, r_near=1.5, w_omega=0.0)


def gate(c, n=(1, 0, 0), h=(0, -1, 0), a=0.75):
    return np.array([[*c, *n, *h, a, a]], dtype=np.float64)


def two_gates():
    return np.vstack([gate((0, 0, 0)), gate((10, 0, 0))])


def seg(P, trk, a, b, g=0, g0=0, front=1, w=(0, 0, 0)):
    return O.gate_paper_step(P, trk, a, b, w, g, g0, front)


def test_progress_is_squared_and_near_term_is_conditional(P):
    trk = O.Track(gates=two_gates())
    # far from the gate (|p - c| = 5 > r_near): progress only, 16 - 25 (eq.(6))
    J, g, _, n = seg(P, trk, (-5, 0, 0), (-4, 0, 0))
    assert J == pytest.approx(16.0 - 25.0, abs=1e-12) and g == 0 and n == 0
    # pre-step state inside r_near: + Q_near |p_k - c|^2 on the PRE-step state (eq.(7) sums p_k)
    J, *_ = seg(P, trk, (-1.0, 0.5, 0), (-0.5, 0.5, 0))
    assert J == pytest.approx((0.25 + 0.25) - (1.0 + 0.25) + 2.0 * 1.25, abs=1e-12)
    # the post-step state being inside does not matter
    J, *_ = seg(P, trk, (-2.0, 0, 0), (-1.0, 0, 0))
    assert J == pytest.approx(1.0 - 4.0, abs=1e-12)
    # threshold is strict: exactly at r_near the term is off; the margin reports the distance to it
    J, _, m, _ = seg(P, trk, (-1.5, 0, 0), (-1.4, 0, 0))
    assert J == pytest.approx(1.96 - 2.25, abs=1e-12) and m == pytest.approx(0.0, abs=1e-15)
    J, _, m, _ = seg(P, trk, (-1.49, 0, 0), (-1.4, 0, 0))
    assert J == pytest.approx(1.96 - 1.49 ** 2 + 2.0 * 1.49 ** 2, abs=1e-12) and m == pytest.approx(0.01, abs=1e-12)


def test_body_rate_term_uses_post_step_rates():
    P = W.base_params(objective=W.OBJ_GATE_PAPER, w_omega=0.01)
    trk = O.Track(gates=two_gates())
    J, *_ = seg(P, trk, (-5, 0, 0), (-4, 0, 0), w=(1, 2, 3))
    assert J == pytest.approx(-9.0 + np.float32(0.01) * 14.0, abs=1e-12)


def test_temporal_check_gates_the_switch(P):
    P = dict(P, gate_pass_bonus=5.0, gate_miss_penalty=10.0, r_near=0.0)
    trk = O.Track(gates=two_gates())
    a, b = (-0.5, 0.1, 0.1), (0.5, 0.1, 0.1)
    prog = (0.25 + 0.02) - (0.25 + 0.02)
    # previous iteration in front at this index: the pass registers (bonus, switch)
    J, g, _, n = seg(P, trk, a, b, front=1)
    assert J == pytest.approx(prog - 5.0, abs=1e-12) and g == 1 and n == 1
    # previous iteration NOT in front: geometric pass of the start gate is ignored (Fig. 2)
    J, g, _, n = seg(P, trk, a, b, front=0)
    assert J == pytest.approx(prog, abs=1e-12) and g == 0 and n == 0
    # a later gate of the horizon (target != start gate) switches on geometry alone [R-25]
    trk3 = O.Track(gates=np.vstack([gate((-20, 0, 0)), gate((0, 0, 0)), gate((10, 0, 0))]))
    J, g, _, n = seg(P, trk3, a, b, g=1, g0=0, front=0)
    assert J == pytest.approx(prog - 5.0, abs=1e-12) and g == 2 and n == 1
    # a crossing outside the opening is a miss whatever the flag says; the target stays
    for front in (0, 1):
        J, g, _, n = seg(P, trk, (-0.5, 0.9, 0), (0.5, 0.9, 0), front=front)
        assert J == pytest.approx(10.0, abs=1e-12) and g == 0 and n == 0
    # back-to-front motion and starting on the plane are no crossings
    assert seg(P, trk, (0.5, 0, 0), (-0.5, 0, 0))[1] == 0
    assert seg(P, trk, (0.0, 0, 0), (0.5, 0, 0))[1] == 0
    # the last gate wraps to the first
    J, g, *_ = seg(P, trk, (9.5, 0, 0), (10.5, 0, 0), g=1, g0=0)
    assert g == 0


def test_rollout_telescopes_without_events():
    # no gate event, near term off: J = |p_N - c|^2 - |p_0 - c|^2 + w sum |omega|^2
    wl = W.cfg0(K=4, N=12)
    p = dict(wl.params, objective=W.OBJ_GATE_PAPER, q_near=0.0, r_near=0.0)
    trk = O.Track(gates=wl.gates)
    r = O.step(p, trk, wl.x0, wl.start, wl.u_nom, 3, 0, want_du=True)
    c = wl.gates[0, 0:3].astype(np.float64)
    for k in range(4):
        x = wl.x0[0].astype(np.float64); acc = 0.0
        for t in range(12):
            T = wl.u_nom[0, t].astype(np.float64) + r["du"][0, k, t]
            x = O.rk4_step(p, x, T)
            acc += p["w_omega"] * np.sum(x[10:13] ** 2)
        expect = np.sum((x[0:3] - c) ** 2) - np.sum((wl.x0[0, 0:3].astype(np.float64) - c) ** 2) + acc
        assert r["ncross"][0, k] == 0
        assert r["cost"][0, k] == pytest.approx(expect, rel=1e-12, abs=1e-11)


def test_front_flags_free_fall_closed_form():
    # T = 0 from rest at height z0 above a horizontal gate plane with normal -z: the state is "in
    # front" (n.(p - c) < 0) while z0 - g t^2 / 2 > z_gate, i.e. for k dt < sqrt(2 (z0 - zg) / g)
    p = W.base_params(N=40, objective=W.OBJ_GATE_PAPER)
    g = np.array([[0, 0, 1.0, 0, 0, -1, 1, 0, 0, 5, 5]], dtype=np.float64)
    trk = O.Track(gates=g)
    x0 = np.zeros(13); x0[2] = 2.0; x0[3] = 1.0
    f, m = O.front_flags(p, trk, x0, 0, np.zeros((40, 4)))
    t_hit = np.sqrt(2 * 1.0 / p["g"])
    k = np.arange(41)
    np.testing.assert_array_equal(f, (k * p["dt"] < t_hit).astype(np.int32))
    assert f[0] == 1 and f[-1] == 0
    s = 1.0 - 0.5 * p["g"] * (k * p["dt"]) ** 2          # = -(n.(p-c)) ; margin = min |s|
    assert m == pytest.approx(np.abs(s).min(), rel=1e-9)
    # hover in front of a vertical gate: every state stays in front
    wl = W.cfg0(N=10)
    f, _ = O.front_flags(dict(wl.params, objective=W.OBJ_GATE_PAPER), O.Track(gates=wl.gates), wl.x0[0], 0, wl.u_nom[0])
    assert f.tolist() == [1] * 11


def _as_dict_track(wl):
    return dict(gates=wl.gates.astype(np.float64), ref=None, path=None, closed=True,
                prev_front=wl.prev_front)


@pytest.mark.parametrize("name,kw", [("gate_paper", dict(K=8, N=3)), ("gate_paper", dict(K=4, N=25)),
                                     ("stress_gate_paper", dict(K=24, N=30))])
def test_brute_force_definition(name, kw):
    wl = W.ALL[name](**kw)
    trk = O.Track(gates=wl.gates, prev_front=wl.prev_front)
    r = O.step(wl.params, trk, wl.x0, wl.start, wl.u_nom, 11, 3, want_du=True)
    J, w, un, du = D.mppi_step(wl.params, _as_dict_track(wl), wl.x0[0].astype(np.float64),
                               int(wl.start[0]), wl.u_nom[0].astype(np.float64), 11, 3)
    np.testing.assert_allclose(r["cost"][0], J, rtol=1e-12, atol=1e-11)
    np.testing.assert_allclose(r["du"][0], du, rtol=0, atol=1e-14)
    np.testing.assert_allclose(r["weights"][0], w, rtol=1e-9, atol=1e-15)
    np.testing.assert_allclose(r["u_new"][0], un, rtol=0, atol=1e-12)


def test_stress_case_exercises_registered_and_ignored_passes():
    wl = W.stress_gate_paper(K=256, N=30)
    trk = O.Track(gates=wl.gates, prev_front=wl.prev_front)
    r = O.step(wl.params, trk, wl.x0, wl.start, wl.u_nom, wl.seed, 0)
    allf = O.step(wl.params, O.Track(gates=wl.gates), wl.x0, wl.start, wl.u_nom, wl.seed, 0)
    reg, geo = r["ncross"][0] > 0, allf["ncross"][0] > 0
    assert reg.sum() >= 20 and (geo & ~reg).sum() >= 20          # some passes registered, some ignored
    assert not (reg & ~geo).any()                               # the flags can only remove passes
    assert (wl.prev_front == 0).any() and (wl.prev_front == 1).any()


# ---- the second reading of eq.(7)'s near term [R-40] (near_mode = 1): "prevent states near the current
# gate p0_gate ... from deviating too much from it" -- the distance is to the horizon's START gate, also after the
# target has switched to the next one.

def test_near_term_against_the_start_gate_after_the_switch(P):
    trk = O.Track(gates=two_gates())                  # gate 0 at the origin, gate 1 at x = 10, normals +x
    P1 = dict(P, near_mode=1)
    # a state 0.5 m BEHIND gate 0 that already targets gate 1 (g = 1, g0 = 0): its own target is 9.5 m away
    a, b = (0.5, 0.25, 0.0), (1.0, 0.25, 0.0)
    prog = ((1.0 - 10.0) ** 2 + 0.0625) - ((0.5 - 10.0) ** 2 + 0.0625)         # eq.(6) against gate 1
    J0, *_ = seg(P, trk, a, b, g=1, g0=0)
    J1, *_ = seg(P1, trk, a, b, g=1, g0=0)
    assert J0 == pytest.approx(prog, abs=1e-12)                               # [R-24]: the term is dead here
    assert J1 == pytest.approx(prog + 2.0 * (0.25 + 0.0625), abs=1e-12)       # [R-40]: Q_near |p_k - c_0|^2
    # before the switch (g = g0) the two readings are the same number
    for a2, b2 in (((-1.0, 0.5, 0), (-0.5, 0.5, 0)), ((-5, 0, 0), (-4, 0, 0))):
        assert seg(P, trk, a2, b2)[0] == seg(P1, trk, a2, b2)[0]
    # beyond r_near of the START gate nothing is added, however close the own target is
    J1, *_ = seg(P1, trk, (9.0, 0, 0), (9.5, 0, 0), g=1, g0=0)
    assert J1 == pytest.approx(0.25 - 1.0, abs=1e-12)
    J0, *_ = seg(P, trk, (9.0, 0, 0), (9.5, 0, 0), g=1, g0=0)
    assert J0 == pytest.approx(0.25 - 1.0 + 2.0 * 1.0, abs=1e-12)             # [R-24] measures against gate 1 there
    # the margin follows the gate the term is measured against: | |p_k - c_0| - r_near |
    *_, mg, _ = O.gate_paper_step(P1, trk, (1.4, 0, 0), (1.6, 0, 0), (0, 0, 0), 1, 0, 1)
    assert mg == pytest.approx(0.1, abs=1e-12)
    # the step that registers the pass of gate 0 still measures its pre-step state against gate 0 in both readings
    Ja, ga, *_ = seg(P, trk, (-0.5, 0, 0), (0.5, 0, 0))
    Jb, gb, *_ = seg(P1, trk, (-0.5, 0, 0), (0.5, 0, 0))
    assert ga == gb == 1 and Ja == Jb


@pytest.mark.parametrize("name,kw", [("gate_paper", dict(K=4, N=25)), ("stress_gate_paper", dict(K=24, N=30))])
def test_brute_force_definition_near_mode_1(name, kw):
    wl = W.ALL[name](**kw)
    wl.params["near_mode"] = 1
    trk = O.Track(gates=wl.gates, prev_front=wl.prev_front)
    r = O.step(wl.params, trk, wl.x0, wl.start, wl.u_nom, 11, 3)
    J, w, un, du = D.mppi_step(wl.params, _as_dict_track(wl), wl.x0[0].astype(np.float64),
                               int(wl.start[0]), wl.u_nom[0].astype(np.float64), 11, 3)
    np.testing.assert_allclose(r["cost"][0], J, rtol=1e-12, atol=1e-11)
    r0 = O.step(dict(wl.params, near_mode=0), trk, wl.x0, wl.start, wl.u_nom, 11, 3)
    if name == "stress_gate_paper":                 # passes happen: the two readings really differ on those samples
        passed = r["ncross"][0] > 0
        assert passed.any() and (np.abs(r["cost"][0] - r0["cost"][0])[passed] > 1e-6).any()
        assert np.array_equal(r["cost"][0][~passed], r0["cost"][0][~passed])
