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
