"""Pins P3-P8: the oracle's f_dyn (eq.(2), torque map PAPER.md:70)
and its RK4 discretisation against closed forms and conservation laws."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2509_14726_b200 import workloads as W


@pytest.fixture(scope="module")
def P():
    p = W.base_params()
    p["lambda"] = 1.0
    return p


def level(p=(0, 0, 0), v=(0, 0, 0), w=(0, 0, 0)):
    x = np.zeros(13); x[0:3] = p; x[3] = 1; x[7:10] = v; x[10:13] = w
    return x


def roll(P, x, T, n):
    xs = [x]
    for _ in range(n):
        xs.append(O.rk4_step(P, xs[-1], T))
    return np.array(xs)


def test_hover_is_an_equilibrium(P):
    # P3: T_i = m g / 4 from rest, level: the state does not move
    hover = P["mass"] * P["g"] / 4
    x0 = level((1, 2, 3))
    xs = roll(P, x0, [hover] * 4, 50)
    assert np.abs(xs - x0).max() < 1e-13


def test_free_fall_closed_form(P):
    # P4: T = 0 -> p = p0 + v0 t - g t^2/2, v = v0 - g t; RK4 is exact for polynomials
    x0 = level((1, -2, 30), (3, -1, 2))
    xs = roll(P, x0, [0, 0, 0, 0], 50)
    t = np.arange(51) * P["dt"]
    g = np.array([0, 0, -P["g"]])
    np.testing.assert_allclose(xs[:, 0:3], x0[0:3] + np.outer(t, x0[7:10]) + 0.5 * np.outer(t ** 2, g),
                               atol=1e-12)
    np.testing.assert_allclose(xs[:, 7:10], x0[7:10] + np.outer(t, g), atol=1e-12)
    np.testing.assert_allclose(xs[:, 3:7], np.tile([1, 0, 0, 0], (51, 1)), atol=0)


def test_vertical_thrust_acceleration(P):
    # level attitude, equal thrusts S: constant a_z = S/m - g, no rotation
    T = [3.0] * 4
    xs = roll(P, level(), T, 20)
    a = 12.0 / P["mass"] - P["g"]
    t = np.arange(21) * P["dt"]
    np.testing.assert_allclose(xs[:, 2], 0.5 * a * t ** 2, atol=1e-13)
    np.testing.assert_allclose(xs[:, 9], a * t, atol=1e-13)
    assert np.abs(xs[:, [0, 1, 7, 8, 10, 11, 12]]).max() == 0


def test_yaw_torque_closed_form(P):
    # P6: T = (a,b,a,b): tau_x = tau_y = 0, omega_z = 2 c_tau (a-b) t / J_z, yaw psi = alpha t^2/2
    a, b = 2.2, 2.0
    xs = roll(P, level(), [a, b, a, b], 50)
    t = np.arange(51) * P["dt"]
    alpha = 2 * P["c_tau"] * (a - b) / P["Jz"]
    np.testing.assert_allclose(xs[:, 12], alpha * t, rtol=0, atol=1e-12)
    assert np.abs(xs[:, 10:12]).max() == 0
    psi = 0.5 * alpha * t ** 2
    np.testing.assert_allclose(xs[:, 3], np.cos(psi / 2), atol=2e-9)
    np.testing.assert_allclose(xs[:, 6], np.sin(psi / 2), atol=2e-9)
    assert np.abs(xs[:, 4:6]).max() == 0
    # thrust stays vertical: p_z has the closed form of a constant vertical acceleration
    az = (2 * a + 2 * b) / P["mass"] - P["g"]
    np.testing.assert_allclose(xs[:, 2], 0.5 * az * t ** 2, atol=1e-12)
    # sign: T1 - T2 + T3 - T4 > 0 gives positive yaw rate (third row)
    assert xs[-1, 12] > 0


def test_roll_and_pitch_torque_maps(P):
    # P7: T=(a,a,b,b) -> only omega_x = sqrt(2)/2 ... = (l/sqrt2)*2(a-b)/Jx * t; T=(b,a,a,b) -> only omega_y
    a, b = 2.3, 2.0
    lever = P["arm"] / np.sqrt(2)
    x1 = O.rk4_step(P, level(), [a, a, b, b])
    assert x1[10] == pytest.approx(lever * 2 * (a - b) / P["Jx"] * P["dt"], rel=1e-12)
    assert x1[11] == 0 and x1[12] == 0
    x1 = O.rk4_step(P, level(), [b, a, a, b])
    assert x1[11] == pytest.approx(lever * 2 * (a - b) / P["Jy"] * P["dt"], rel=1e-12)
    assert x1[10] == 0 and x1[12] == 0
    # literal signs of PAPER.md:70: tau_x = l/sqrt2 (T1+T2-T3-T4), tau_y = l/sqrt2 (-T1+T2+T3-T4)
    d = O.fdyn(P, level(), [1, 0, 0, 0])
    assert d[10] > 0 and d[11] < 0 and d[12] > 0
    d = O.fdyn(P, level(), [0, 0, 0, 1])
    assert d[10] < 0 and d[11] < 0 and d[12] < 0


def test_torque_free_precession(P):
    # P8: equal thrusts, omega0 = (wx,0,wz), Jx = Jy: omega_z constant, (wx,wy) rotates at
    # Omega = (Jz - Jx)/Jx * wz; |J omega| and kinetic energy conserved
    hover = P["mass"] * P["g"] / 4
    wx, wz = 3.0, 8.0
    xs = roll(P, level(w=(wx, 0, wz)), [hover] * 4, 50)
    t = np.arange(51) * P["dt"]
    Om = (P["Jz"] - P["Jx"]) / P["Jx"] * wz
    np.testing.assert_allclose(xs[:, 12], wz, atol=1e-12)
    # RK4 truncation: 50 steps x (Om dt)^5/120 x |wx| ~ 2e-5; a wrong sign gives O(1)
    np.testing.assert_allclose(xs[:, 10], wx * np.cos(Om * t), atol=5e-5)
    np.testing.assert_allclose(xs[:, 11], wx * np.sin(Om * t), atol=5e-5)
    Jv = np.array([P["Jx"], P["Jy"], P["Jz"]])
    Lmag = np.linalg.norm(xs[:, 10:13] * Jv, axis=1)
    E = 0.5 * np.sum(xs[:, 10:13] ** 2 * Jv, axis=1)
    assert np.abs(Lmag - Lmag[0]).max() < 1e-7 * Lmag[0]      # RK4 drift ~3e-8 over 50 steps
    assert np.abs(E - E[0]).max() < 2e-7 * E[0]


def test_quaternion_kinematics_constant_body_rate(P):
    # constant omega about body x with Jy = Jx, no torque: q = (cos(w t/2), sin(w t/2), 0, 0)
    hover = P["mass"] * P["g"] / 4
    w = 4.0
    xs = roll(P, level(w=(w, 0, 0)), [hover] * 4, 40)
    t = np.arange(41) * P["dt"]
    np.testing.assert_allclose(xs[:, 3], np.cos(w * t / 2), atol=1e-7)   # RK4 phase error 40 (w dt/2)^5/120
    np.testing.assert_allclose(xs[:, 4], np.sin(w * t / 2), atol=1e-7)
    # body z tilts towards -y for a positive roll: a_y = -(S/m) sin(w t) < 0
    assert xs[10, 8] < 0


def test_thrust_direction_follows_attitude(P):
    # 90 deg pitch about body y: body z points along world +x; acceleration = S/m along x
    q = [np.cos(np.pi / 4), 0, np.sin(np.pi / 4), 0]
    x = level(); x[3:7] = q
    d = O.fdyn(P, x, [1, 1, 1, 1])
    np.testing.assert_allclose(d[7:10], [4 / P["mass"], 0, -P["g"]], atol=1e-12)
    # 90 deg roll about body x: body z points along world -y
    x[3:7] = [np.cos(np.pi / 4), np.sin(np.pi / 4), 0, 0]
    d = O.fdyn(P, x, [1, 1, 1, 1])
    np.testing.assert_allclose(d[7:10], [0, -4 / P["mass"], -P["g"]], atol=1e-12)


def test_quaternion_norm_is_preserved(P):
    # P5: |q| = 1 to 1e-9 after every step, here under violent tumbling
    rng = np.random.default_rng(0)
    x = level(w=(30, -40, 10))
    for _ in range(200):
        x = O.rk4_step(P, x, rng.uniform(0, 7, 4))
        assert abs(np.linalg.norm(x[3:7]) - 1) < 1e-12


def test_rk4_is_fourth_order(P):
    # halving dt must cut the one-step-pair error ~16x against a fine reference
    x0 = level(w=(5, -3, 2), v=(1, 2, 3)); x0[3:7] = np.array([0.9, 0.1, -0.3, 0.2]) / np.linalg.norm([0.9, 0.1, -0.3, 0.2])
    T = [1.0, 3.0, 2.0, 4.0]

    def run(n, tot=0.08):
        x = x0
        for _ in range(n):
            x = O.rk4_step(P, x, T, tot / n)
        return x
    ref = run(512)
    e1 = np.abs(run(2) - ref).max(); e2 = np.abs(run(4) - ref).max()
    assert 10 < e1 / e2 < 24
