"""Host side of the closed-loop lap experiment (paper_2509_14726_b200/closed_loop.py): the reductions of
a flight log are checked on hand-built trajectories with known answers."""
import numpy as np
import pytest

from paper_2509_14726_b200 import closed_loop as CL
from paper_2509_14726_b200 import workloads as W


def circle_log(radius, speed, dt, steps, z=1.5, B=1, phase=-0.4):
    t = np.arange(steps + 1) * dt
    ang = phase + speed / radius * t
    x = np.zeros((steps + 1, B, 13), np.float32)
    x[:, :, 0] = (radius * np.cos(ang))[:, None]; x[:, :, 1] = (radius * np.sin(ang))[:, None]; x[:, :, 2] = z
    x[:, :, 3] = 1.0
    x[:, :, 7] = (-speed * np.sin(ang))[:, None]; x[:, :, 8] = (speed * np.cos(ang))[:, None]
    return CL.FlightLog(x, np.zeros((steps + 1, B), np.int32), dt)


def test_gate_passes_and_lap_time_on_a_circle():
    gates = W.circle_gates().astype(np.float64)          # 4 gates, radius 5, normals tangent (counter-clockwise)
    R, v, dt = 5.2, 8.0, 0.02                            # flown 0.2 m outside the gate centres
    log = circle_log(R, v, dt, 1200)
    m = CL.lap_metrics(log, gates, laps=3)[0]
    # gate 0 sits at angle 0: first pass after 0.4 rad, then every quarter turn
    omega = v / R
    assert m["passes"] == int((1200 * dt * omega - 0.4) / (np.pi / 2)) + 1
    assert m["flight_time_s"] == pytest.approx((0.4 + 11 * np.pi / 2) / omega, abs=2e-3)   # 12th pass
    assert m["wp_dist_min"] == pytest.approx(0.2, abs=2e-3) and m["wp_dist_max"] == pytest.approx(0.2, abs=2e-3)
    assert m["speed_mean"] == pytest.approx(v, rel=1e-6)
    # too far out: outside the 1.5 m opening -> no pass at all
    far = CL.lap_metrics(circle_log(6.0, v, dt, 600), gates, laps=1)[0]
    assert far["passes"] == 0 and far["flight_time_s"] is None
    # flying the circle backwards crosses every plane back to front: no pass
    back = circle_log(R, -v, dt, 600)
    assert CL.lap_metrics(back, gates, laps=1)[0]["passes"] == 0


def test_passes_follow_the_gate_order():
    gates = W.circle_gates().astype(np.float64)
    p = np.array([[5.0, -1.0, 1.5], [5.0, 1.0, 1.5],          # through gate 0 (normal +y at (5,0))
                  [5.0, -1.0, 1.5], [5.0, 1.0, 1.5],          # gate 0 again: not the current target -> ignored
                  [1.0, 5.0, 1.5], [-1.0, 5.0, 1.5]])         # gate 1 at (0,5), normal -x
    out = CL.gate_passes(p, gates)
    assert [(t, g) for t, g, _, _ in out] == [(1, 0), (5, 1)]
    assert out[0][2] == pytest.approx(0.0, abs=1e-12) and out[0][3] == pytest.approx(0.5)


def test_tracking_rmse_and_contour_rms():
    ref = np.zeros((101, 13)); ref[:, 0] = np.linspace(0, 10, 101)
    x = np.zeros((101, 2, 13), np.float32); x[:, :, 0] = ref[:, None, 0]
    x[:, 1, 1] = 0.3; x[:, 1, 2] = 0.4                        # drone 1 flies 0.5 m off
    log = CL.FlightLog(x, np.zeros((101, 2), np.int32), 0.02)
    np.testing.assert_allclose(CL.tracking_rmse(log, ref), [0.0, 0.5], atol=1e-6)
    ang = np.linspace(0, 2 * np.pi, 400, endpoint=False)
    path = np.stack([5 * np.cos(ang), 5 * np.sin(ang), np.full_like(ang, 1.5)], 1)
    flown = circle_log(5.3, 6.0, 0.02, 500)
    assert CL.contour_rms(flown, path)[0] == pytest.approx(0.3, abs=2e-3)


def test_lap_workloads_are_well_formed():
    for kind in ("gate", "gate_paper", "track", "contour"):
        wl = W.lap(kind, B=3, K=64, N=10, steps=20)
        assert wl.x0.shape == (3, 13) and wl.u_nom.shape == (3, 10, 4) and wl.params["B"] == 3
        if kind == "track":
            assert wl.ref.shape[0] >= 20 + 10 + 1


def test_progress_metrics_on_a_square_path():
    # rows of 19 (objective 4): the vehicle runs 0.3 m beside a 4 x 4 m square path at 4 m/s while its
    # progress state theta advances at exactly that speed: laps, lap times and the distance between the
    # vehicle and P(theta) have closed forms
    path = np.array([[0, 0, 1], [4, 0, 1], [4, 4, 1], [0, 4, 1]], np.float32)      # closed, L = 16
    dt, steps, v = 0.02, 500, 4.0
    t = np.arange(steps + 1) * dt
    th = 1.0 + v * t                                        # theta_0 = 1 m
    s = np.mod(th, 16.0)
    on = np.stack([np.select([s < 4, s < 8, s < 12], [s, 4 + 0 * s, 12 - s], 0 * s),
                   np.select([s < 4, s < 8, s < 12], [0 * s, s - 4, 4 + 0 * s], 16 - s), np.ones_like(s)], 1)
    x = np.zeros((steps + 1, 2, 19), np.float32)
    x[:, 0, 0:3] = on + [0, 0, 0.3]                         # drone 0: 0.3 m above P(theta)
    x[:, 1, 0:3] = on                                       # drone 1: exactly on it ...
    x[:, :, 7] = v; x[:, :, 17] = th[:, None]
    x[:, 1, 17] = 1.0 + 0.5 * v * t                         # ... but its theta runs at half the speed
    log = CL.FlightLog(x, np.zeros((steps + 1, 2), np.int32), dt)
    m0, m1 = CL.progress_metrics(log, path)
    assert m0["progress_m"] == pytest.approx(v * steps * dt, abs=1e-4) and m0["laps"] == pytest.approx(40.0 / 16.0, abs=1e-5)
    np.testing.assert_allclose(m0["lap_times_s"], [4.0, 8.0], atol=dt)
    assert m0["dist_to_progress_point_max"] == pytest.approx(0.3, abs=1e-5)
    assert m0["speed_mean"] == pytest.approx(v)
    assert m1["laps"] == pytest.approx(20.0 / 16.0, abs=1e-5) and len(m1["lap_times_s"]) == 1
    assert m1["dist_to_progress_point_max"] > 3.9          # the vehicle ran away from its progress point
    # contour_rms sees the same flights: 0.3 m beside the path / on it
    np.testing.assert_allclose(CL.contour_rms(log, path), [0.3, 0.0], atol=1e-5)


def test_replicate_keeps_every_array_consistent():
    for name in ("cfg1", "gate_paper", "contour_paper"):
        base = W.ALL[name](K=64, N=8)
        wl = W.replicate(base, 5, jitter=0.2)
        assert wl.params["B"] == 5 and wl.x0.shape == (5, base.x0.shape[1]) and wl.u_nom.shape == (5, 8, 4)
        assert np.abs(wl.x0[:, 0:3] - base.x0[0, 0:3]).max() <= 0.2 + 1e-6 and np.ptp(wl.x0[:, 0]) > 0
        np.testing.assert_array_equal(wl.x0[:, 3:], np.repeat(base.x0[:, 3:], 5, 0))
        assert (wl.v_nom is None) == (base.v_nom is None) and (wl.prev_front is None) == (base.prev_front is None)
        if wl.v_nom is not None:
            assert wl.v_nom.shape == (5, 8)
        assert base.params["B"] == 1                                  # the original is untouched
