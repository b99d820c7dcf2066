"""Pins P10, P12, P13: the three objectives of the oracle on hand-built cases.
Gate progress eq.(6) PAPER.md:105-112 with BASELINE.json configs[0] constants; tracking eq.(8)
PAPER.md:139-147; contouring eq.(9) PAPER.md:149-161 in the projection variant of configs[3]."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2509_14726_b200 import workloads as W


@pytest.fixture(scope="module")
def P():
    return W.base_params()


def gate(c, n=(1, 0, 0), h=(0, -1, 0), a=0.75):
    # n = +x, h = (n_y, -n_x, 0) = (0,-1,0), v = h x n = +z
    return list(c) + list(n) + list(h) + [a, a]


# ---- P10: gate logic on single straight segments, gate at the origin, normal +x -----------

def seg(P, trk, a, b, g=0, w=(0, 0, 0)):
    return O.gate_step(P, trk, a, b, w, g)


def test_gate_pass_through_centre(P):
    trk = O.Track(gates=[gate((0, 0, 0)), gate((10, 0, 0))])
    J, g, margin, nc = seg(P, trk, (-1, 0, 0), (1, 0, 0))
    assert J == pytest.approx(1.0 - 1.0 - 5.0) and g == 1 and nc == 1


def test_gate_opening_edges(P):
    trk = O.Track(gates=[gate((0, 0, 0)), gate((10, 0, 0))])
    for off, ok in ((0.74, True), (0.76, False), (-0.74, True), (-0.76, False), (0.75, True)):
        J, g, _, _ = seg(P, trk, (-1, off, 0), (1, off, 0))
        assert (g == 1) == ok
        assert J == pytest.approx(-5.0 if ok else 10.0)
        J, g, _, _ = seg(P, trk, (-1, 0, off), (1, 0, off))
        assert (g == 1) == ok
        assert J == pytest.approx(-5.0 if ok else 10.0)


def test_gate_crossing_point_is_interpolated(P):
    # oblique segment: y goes 0.5 -> 1.5 while x goes -1 -> 3; plane hit at alpha = 1/4: y = 0.75
    trk = O.Track(gates=[gate((0, 0, 0)), gate((10, 0, 0))])
    _, g, margin, _ = seg(P, trk, (-1, 0.5, 0), (3, 1.5, 0))
    assert g == 1 and margin == pytest.approx(0.0, abs=1e-15)
    _, g, _, _ = seg(P, trk, (-1, 0.5, 0), (3, 1.5 + 1e-6, 0))
    assert g == 0


def test_gate_plane_boundary_cases(P):
    trk = O.Track(gates=[gate((0, 0, 0)), gate((10, 0, 0))])
    # ends exactly on the plane: counts
    J, g, _, _ = seg(P, trk, (-1, 0, 0), (0, 0, 0))
    assert g == 1 and J == pytest.approx(0 - 1 - 5)
    # starts on the plane: no crossing
    J, g, _, _ = seg(P, trk, (0, 0, 0), (1, 0, 0))
    assert g == 0 and J == pytest.approx(1.0)
    # back to front: no crossing, no penalty
    J, g, _, _ = seg(P, trk, (1, 0, 0), (-1, 0, 0))
    assert g == 0 and J == pytest.approx(0.0)
    # stays in front
    J, g, m, _ = seg(P, trk, (-3, 0, 0), (-1, 0, 0))
    assert g == 0 and J == pytest.approx(-2.0) and m == pytest.approx(1.0)


def test_gate_only_current_gate_registers_and_wraps(P):
    # two gates 0.1 m apart crossed in one step: only gate 0 registers; progress wholly vs gate 0
    trk = O.Track(gates=[gate((0, 0, 0)), gate((0.1, 0, 0))])
    J, g, _, nc = seg(P, trk, (-1, 0, 0), (1, 0, 0), g=0)
    assert g == 1 and nc == 1 and J == pytest.approx(-5.0)
    # next step against gate 1 (already behind it): nothing happens
    J, g, _, _ = seg(P, trk, (1, 0, 0), (2, 0, 0), g=1)
    assert g == 1 and J == pytest.approx(1.9 - 0.9)
    # last gate wraps to 0
    J, g, _, _ = seg(P, trk, (-1, 0, 0), (1, 0, 0), g=1)
    assert g == 0


def test_gate_miss_keeps_target_and_body_rate_term(P):
    trk = O.Track(gates=[gate((0, 0, 0)), gate((10, 0, 0))])
    J, g, _, nc = seg(P, trk, (-1, 2, 0), (1, 2, 0), w=(1, 2, 3))
    assert g == 0 and nc == 0
    assert J == pytest.approx(10.0 + P["w_omega"] * 14.0)


def test_gate_rotated_frame(P):
    # gate with normal +y, h = (1,0,0), v = h x n = +z; half-width 0.5 along h, half-height 1 along v
    g0 = [2, 3, 1, 0, 1, 0, 1, 0, 0, 0.5, 1.0]
    trk = O.Track(gates=[g0, g0])
    assert seg(P, trk, (2.4, 2, 1.9), (2.4, 4, 1.9))[1] == 1
    assert seg(P, trk, (2.6, 2, 1.0), (2.6, 4, 1.0))[1] == 0      # outside along h
    assert seg(P, trk, (2.0, 2, 2.1), (2.0, 4, 2.1))[1] == 0      # outside along v


def test_gate_telescoping_without_events(P):
    # P10(ix): no event => J = d_N - d_0 + w_omega sum |omega|^2 (full oracle rollout, sigma = 0)
    wl = W.cfg0(K=32, N=20)
    p = dict(wl.params); p["sigma"] = 0.0
    u = wl.u_nom.astype(np.float64).copy(); u[0, :, :] += 0.3      # climb, no rotation
    r = O.step(p, O.Track(gates=wl.gates), wl.x0, wl.start, u, 0, 0)
    c = wl.gates[0, 0:3].astype(np.float64)
    x = wl.x0[0].astype(np.float64)
    d0 = np.linalg.norm(x[0:3] - c)
    for t in range(20):
        x = O.rk4_step(p, x, u[0, t])
    assert r["ncross"].max() == 0
    np.testing.assert_allclose(r["cost"][0], np.linalg.norm(x[0:3] - c) - d0, rtol=0, atol=1e-12)


# ---- P12: tracking ------------------------------------------------------------------------

def test_tracking_terms(P):
    rng = np.random.default_rng(1)
    x = rng.normal(size=13); x[3:7] /= np.linalg.norm(x[3:7])
    xr = rng.normal(size=13); xr[3:7] /= np.linalg.norm(xr[3:7])
    J = O.track_state_term(P, x, xr)
    qd = abs(x[3:7] @ xr[3:7])
    want = (P["Qp"] * np.sum((x[0:3] - xr[0:3]) ** 2) + P["Qv"] * np.sum((x[7:10] - xr[7:10]) ** 2)
            + P["Qw"] * np.sum((x[10:13] - xr[10:13]) ** 2) + P["Qq"] * (2 - 2 * qd))
    assert J == pytest.approx(want, rel=1e-13)
    # q and -q are the same attitude
    x2 = x.copy(); x2[3:7] *= -1
    assert O.track_state_term(P, x2, xr) == pytest.approx(J, rel=1e-14)
    assert O.track_state_term(P, xr, xr) == 0.0
    # each weight acts on its own block
    for sl, key in ((slice(0, 3), "Qp"), (slice(7, 10), "Qv"), (slice(10, 13), "Qw")):
        y = xr.copy(); y[sl] += [1, 2, 2]
        assert O.track_state_term(P, y, xr) == pytest.approx(9 * P[key], rel=1e-13)
    hover = P["mass"] * P["g"] / 4
    T = hover + np.array([0.1, -0.2, 0.3, 0.0])
    assert O.track_stage(P, xr, T, xr) == pytest.approx(P["R"] * 0.14, rel=1e-9)


def test_tracking_rollout_n1(P):
    # x0 = ref[0], N = 1: J = R sum (T - hover)^2 + terminal state term at x_1 vs ref[1]
    wl = W.cfg2(K=32, N=1)
    trk = O.Track(ref=wl.ref)
    r = O.step(wl.params, trk, wl.x0, wl.start, wl.u_nom, 5, 2, want_du=True)
    hover = wl.params["mass"] * wl.params["g"] / 4
    for k in (0, 7, 31):
        T = wl.u_nom[0, 0].astype(np.float64) + r["du"][0, k, 0]
        x1 = O.rk4_step(wl.params, wl.x0[0], T)
        want = wl.params["R"] * np.sum((T - hover) ** 2) + O.track_state_term(wl.params, x1, wl.ref[1])
        assert r["cost"][0, k] == pytest.approx(want, rel=1e-13)


# ---- P13: contouring ----------------------------------------------------------------------

def test_path_prepare_straight_and_circle():
    pts = np.stack([np.arange(10) * 0.5, np.zeros(10), np.ones(10)], axis=1)
    s, tan, L = O.path_prepare(pts, closed=False)
    np.testing.assert_allclose(s, np.arange(10) * 0.5, atol=1e-15)
    np.testing.assert_allclose(tan, np.tile([1, 0, 0], (10, 1)), atol=1e-15)
    assert L == pytest.approx(4.5)
    a = 2 * np.pi * np.arange(400) / 400
    circ = np.stack([3 * np.cos(a), 3 * np.sin(a), np.zeros(400)], axis=1)
    s, tan, L = O.path_prepare(circ, closed=True)
    chord = 2 * 3 * np.sin(np.pi / 400)
    assert L == pytest.approx(400 * chord, rel=1e-12)
    np.testing.assert_allclose(tan, np.stack([-np.sin(a), np.cos(a), 0 * a], axis=1), atol=1e-12)


def test_contour_straight_path_parallel_flight(P):
    # drone flies parallel to a straight path at lateral offset e: e_c^2 = e^2, sum dS = distance
    pts = np.stack([np.arange(200) * 0.05, np.zeros(200), np.zeros(200)], axis=1)
    trk = O.Track(path=pts, closed=False)
    e = 0.3
    idx = O.path_nearest(pts, False, (1.0, e, 0), -1, 16)
    assert idx == 20
    theta = 1.0
    tot = 0.0
    for i in range(1, 30):
        p = (1.0 + 0.11 * i, e, 0)
        J, idx, th = O.contour_step(P, trk, p, (0, 0, 0), idx, theta)
        el = p[0] - pts[idx, 0]
        assert abs(el) <= 0.025 + 1e-12
        assert J == pytest.approx(P["q_contour"] * e * e + P["q_lag"] * el * el
                                  - P["mu_progress"] * (th - theta), rel=1e-12)
        assert th == pytest.approx(p[0], abs=1e-12)
        tot += th - theta; theta = th
    assert tot == pytest.approx(0.11 * 29, abs=1e-12)


def test_contour_circle_radius_offset_and_wrap(P):
    a = 2 * np.pi * np.arange(500) / 500
    R = 5.0
    pts = np.stack([R * np.cos(a), R * np.sin(a), np.zeros(500)], axis=1)
    trk = O.Track(path=pts, closed=True)
    s, tan, L = O.path_prepare(pts, True)
    r = 5.4
    ang0 = -0.05
    idx = O.path_nearest(pts, True, (r * np.cos(ang0), r * np.sin(ang0), 0), -1, 16)
    assert idx == 496
    theta = s[idx] + np.dot(np.array([r * np.cos(ang0), r * np.sin(ang0), 0]) - pts[idx], tan[idx])
    for i in range(1, 12):                       # crosses index 0: progress must stay positive
        ang = ang0 + 0.02 * i
        p = (r * np.cos(ang), r * np.sin(ang), 0)
        J, idx, th = O.contour_step(P, trk, p, (0, 0, 1), idx, theta)
        d = th - theta
        d -= L * np.ceil((d - L / 2) / L)
        assert 0.08 < d < 0.12                   # ~ R * 0.02 = 0.1 of arc per step
        el = np.dot(np.array(p) - pts[idx], tan[idx])
        ec2 = np.sum((np.array(p) - pts[idx]) ** 2) - el ** 2
        assert np.sqrt(ec2) == pytest.approx(r - R, abs=2e-3)
        assert J == pytest.approx(P["q_contour"] * ec2 + P["q_lag"] * el ** 2 - P["mu_progress"] * d
                                  + P["w_omega"], rel=1e-10)
        theta = th


def test_contour_window_equals_global_when_motion_is_small():
    wl = W.cfg3(K=8, N=5)
    pts = wl.path.astype(np.float64)
    rng = np.random.default_rng(2)
    for _ in range(50):
        c = int(rng.integers(0, 500))
        p = pts[c] + rng.normal(scale=0.3, size=3)
        assert O.path_nearest(pts, True, p, c, 16) == O.path_nearest(pts, True, p, -1, 16)
    # first minimiser on an exact tie: midpoint between vertices 10 and 11 of a straight path
    st = np.stack([np.arange(30) * 1.0, np.zeros(30), np.zeros(30)], axis=1)
    assert O.path_nearest(st, False, (10.5, 0, 0), 12, 16) == 10
    assert O.path_nearest(st, False, (10.5, 0, 0), -1, 16) == 10
    # open path: indices outside [0,P-1] are skipped, closed path wraps
    assert O.path_nearest(st, False, (-3, 0, 0), 2, 16) == 0
    assert O.path_nearest(st, True, (29.2, 0, 0), 1, 16) == 29
