"""Pins for the oracle's dynamics (O1, O2), playback (D8) and log divergence (O5).

Each expected value below comes from the paper's equations solved in closed form (or from a
structurally different formula, e.g. the paper's own inverse Eq. 3), never from re-typing
the update the oracle implements.
"""
import math

import numpy as np
import pytest

import oracle
from util import mk_traj, set_agent

DT = 0.1


def _run_bicycle(x, y, yaw, v, acc, kappa, n, B=1):
    """n bicycle steps of one agent with constant (acc, kappa); returns sim dict."""
    T = n + 1
    log = mk_traj(1, T, 1, valid=1)
    sim = mk_traj(1, T, 1, valid=0)
    set_agent(sim, 0, 0, 0, x, y, yaw, v * math.cos(yaw), v * math.sin(yaw))
    act = np.zeros((1, 2, 1), np.float32)
    act[0, 0, 0], act[0, 1, 0] = acc, kappa
    av = np.ones((1, 1), np.uint8)
    for t in range(n):
        oracle.step(log, sim, t, oracle.DYN_BICYCLE, act, av, dt=DT, max_accel=0, max_curvature=0)
    return sim


# P1 (Eq. 2 with kappa=0): the update is the exact constant-acceleration
# integrator along the heading: p_n = p_0 + (cos,sin)(v0 n dt + a (n dt)^2 / 2), v_n = v0 + a n dt.
@pytest.mark.parametrize("yaw,v0,acc", [(0.0, 5.0, 0.0), (0.7, 10.0, 2.0), (-2.1, 3.0, -0.25), (math.pi / 2, 0.0, 3.0)])
def test_bicycle_straight_line_closed_form(yaw, v0, acc):
    n = 40
    sim = _run_bicycle(1.0, -2.0, yaw, v0, acc, 0.0, n)
    for k in (1, 7, n):
        tt = k * DT
        s = v0 * tt + 0.5 * acc * tt * tt
        assert sim["x"][0, k, 0] == pytest.approx(1.0 + math.cos(yaw) * s, abs=2e-5)
        assert sim["y"][0, k, 0] == pytest.approx(-2.0 + math.sin(yaw) * s, abs=2e-5)
        assert sim["yaw"][0, k, 0] == pytest.approx(yaw, abs=1e-7)
        vn = v0 + acc * tt
        assert sim["vel_x"][0, k, 0] == pytest.approx(vn * math.cos(yaw), abs=1e-5)
        assert sim["vel_y"][0, k, 0] == pytest.approx(vn * math.sin(yaw), abs=1e-5)


# P2 (Eq. 2 with a=0, constant kappa, v): yaw_n = yaw_0 + n kappa v dt, and the positions are
# the vertices of a regular polygon inscribed in a circle of radius r = v dt / (2 sin(kappa v dt/2))
# (chord length v dt, turning angle kappa v dt).  For kappa=0.1, v=15: r = 10.00938 m, not 1/kappa.
@pytest.mark.parametrize("kappa,v", [(0.1, 15.0), (-0.05, 8.0), (0.3, 2.0)])
def test_bicycle_constant_curvature_polygon(kappa, v):
    n = 60
    yaw0 = 0.3
    sim = _run_bicycle(3.0, 4.0, yaw0, v, 0.0, kappa, n)
    dth = kappa * v * DT
    r = v * DT / (2.0 * math.sin(abs(dth) / 2.0))
    # Step k moves along heading yaw_k (the position uses v_x, v_y = v(cos,sin)(yaw_k)), so the
    # chord directions are yaw0 + k*dth: polygon centre lies at distance r from every vertex,
    # on the left (kappa>0) of the first chord's perpendicular bisector.
    sgn = 1.0 if kappa > 0 else -1.0
    mid = np.array([3.0 + 0.5 * v * DT * math.cos(yaw0), 4.0 + 0.5 * v * DT * math.sin(yaw0)])
    apothem = r * math.cos(abs(dth) / 2.0)
    centre = mid + sgn * apothem * np.array([-math.sin(yaw0), math.cos(yaw0)])
    px = sim["x"][0, :, 0].astype(np.float64); py = sim["y"][0, :, 0].astype(np.float64)
    rad = np.hypot(px - centre[0], py - centre[1])
    assert np.allclose(rad, r, atol=5e-5), (rad.min(), rad.max(), r)
    if kappa == 0.1:
        assert r == pytest.approx(10.00938, abs=1e-5)
        assert abs(r - 1.0 / kappa) / (1.0 / kappa) == pytest.approx(9.4e-4, rel=0.02)
    assert sim["yaw"][0, n, 0] == pytest.approx(yaw0 + n * dth, abs=1e-5)
    speed = np.hypot(sim["vel_x"][0, :, 0], sim["vel_y"][0, :, 0])
    assert np.allclose(speed, v, atol=1e-5)


def test_bicycle_polygon_closure():
    # n * kappa v dt = 2 pi -> back to the start (regular n-gon), P2.
    n = 48
    v = 10.0
    kappa = 2 * math.pi / (n * v * DT)
    sim = _run_bicycle(0.0, 0.0, 0.0, v, 0.0, kappa, n)
    assert sim["x"][0, n, 0] == pytest.approx(0.0, abs=1e-4)
    assert sim["y"][0, n, 0] == pytest.approx(0.0, abs=1e-4)


# P3: the paper's own inverse (Eq. 3, with atan2(v_y', v_x') per reading D4) applied
# to (s, step(s, a, kappa)) returns (a, kappa).
def test_bicycle_inverse_roundtrip():
    rng = np.random.default_rng(7)
    for _ in range(200):
        yaw = rng.uniform(-1.0, 1.0); v = rng.uniform(1.0, 15.0)
        acc = rng.uniform(-3, 3); kappa = rng.uniform(-0.1, 0.1)
        sim = _run_bicycle(rng.uniform(-50, 50), rng.uniform(-50, 50), yaw, v, acc, kappa, 1)
        vx0, vy0 = float(sim["vel_x"][0, 0, 0]), float(sim["vel_y"][0, 0, 0])
        vx1, vy1 = float(sim["vel_x"][0, 1, 0]), float(sim["vel_y"][0, 1, 0])
        sp0, sp1 = math.hypot(vx0, vy0), math.hypot(vx1, vy1)
        a_inv = (sp1 - sp0) / DT
        k_inv = (math.atan2(vy1, vx1) - float(sim["yaw"][0, 0, 0])) / (sp0 * DT + 0.5 * a_inv * DT * DT)
        assert a_inv == pytest.approx(acc, abs=2e-4)
        assert k_inv == pytest.approx(kappa, abs=2e-5)


def test_bicycle_position_uses_velocity_components_not_yaw():
    # Eq. 2 asymmetry (O1): x' = x + v_x dt + a cos(yaw) dt^2/2.  With velocity perpendicular to
    # the heading the displacement has both parts.
    log = mk_traj(1, 2, 1, valid=1); sim = mk_traj(1, 2, 1)
    set_agent(sim, 0, 0, 0, 0.0, 0.0, 0.0, 0.0, 4.0)      # yaw 0, velocity along +y
    act = np.array([[[2.0], [0.0]]], np.float32); av = np.ones((1, 1), np.uint8)
    oracle.step(log, sim, 0, oracle.DYN_BICYCLE, act, av)
    assert sim["x"][0, 1, 0] == pytest.approx(0.5 * 2.0 * DT * DT, abs=1e-7)   # from a cos(yaw)
    assert sim["y"][0, 1, 0] == pytest.approx(4.0 * DT, abs=1e-7)              # from v_y
    assert sim["vel_x"][0, 1, 0] == pytest.approx(4.0 + 2.0 * DT, abs=1e-6)    # v' along yaw'=0
    assert sim["vel_y"][0, 1, 0] == pytest.approx(0.0, abs=1e-6)


def test_bicycle_negative_speed_and_no_wrap():
    # D6: v' = v + a dt may go negative, velocity then points backwards; D5: yaw is not wrapped.
    sim = _run_bicycle(0.0, 0.0, 3.1, 0.1, -3.0, 0.0, 1)
    assert sim["vel_x"][0, 1, 0] == pytest.approx((0.1 - 0.3) * math.cos(3.1), abs=1e-6)
    sim = _run_bicycle(0.0, 0.0, 3.1, 10.0, 0.0, 0.1, 5)
    assert sim["yaw"][0, 5, 0] == pytest.approx(3.1 + 5 * 0.1 * 10.0 * DT, abs=1e-5)  # > pi


def test_action_clipping_D7():
    # limits 6 m/s^2 and 0.3 1/m: out-of-range actions behave as the clipped ones.
    log = mk_traj(1, 2, 2, valid=1)
    sim = mk_traj(1, 2, 2)
    for a in range(2):
        set_agent(sim, 0, 0, a, 1.0, 2.0, 0.4, 5.0 * math.cos(0.4), 5.0 * math.sin(0.4))
    act = np.array([[[9.0, 6.0], [-0.8, -0.3]]], np.float32)   # agent0 out of range, agent1 at limit
    av = np.ones((1, 2), np.uint8)
    oracle.step(log, sim, 0, oracle.DYN_BICYCLE, act, av, max_accel=6.0, max_curvature=0.3)
    for k in ("x", "y", "yaw", "vel_x", "vel_y"):
        assert sim[k][0, 1, 0] == sim[k][0, 1, 1], k
    sim2 = {k: v.copy() for k, v in sim.items()}
    oracle.step(log, sim2, 0, oracle.DYN_BICYCLE, act, av, max_accel=0, max_curvature=0)   # disabled
    assert sim2["x"][0, 1, 0] != sim2["x"][0, 1, 1]


# P4 (Eq. 1)
def test_delta_local_reduces_to_eq1_at_zero_yaw_and_rotates():
    log = mk_traj(1, 2, 2, valid=1); sim = mk_traj(1, 2, 2)
    set_agent(sim, 0, 0, 0, 10.0, 20.0, 0.0)
    phi = 1.1
    c, s = math.cos(phi), math.sin(phi)
    set_agent(sim, 0, 0, 1, c * 10 - s * 20, s * 10 + c * 20, phi)
    act = np.array([[[0.4, 0.4], [-0.3, -0.3], [0.05, 0.05]]], np.float32)
    av = np.ones((1, 2), np.uint8)
    oracle.step(log, sim, 0, oracle.DYN_DELTA_LOCAL, act, av)
    # yaw = 0: world-frame Eq. 1 literally
    assert sim["x"][0, 1, 0] == pytest.approx(10.4, abs=1e-6)
    assert sim["y"][0, 1, 0] == pytest.approx(19.7, abs=2e-6)
    assert sim["yaw"][0, 1, 0] == pytest.approx(0.05, abs=1e-7)
    assert sim["vel_x"][0, 1, 0] == pytest.approx(4.0, abs=2e-4)     # (x'-x)/dt on float32 state
    assert sim["vel_y"][0, 1, 0] == pytest.approx(-3.0, abs=2e-4)
    # rotating the initial state by phi rotates the output by phi
    x1, y1 = c * 10.4 - s * 19.7, s * 10.4 + c * 19.7
    assert sim["x"][0, 1, 1] == pytest.approx(x1, abs=5e-6)
    assert sim["y"][0, 1, 1] == pytest.approx(y1, abs=5e-6)
    assert sim["yaw"][0, 1, 1] == pytest.approx(phi + 0.05, abs=2e-7)


def test_delta_local_straight_along_heading():
    log = mk_traj(1, 6, 1, valid=1); sim = mk_traj(1, 6, 1)
    yaw = 2.2
    set_agent(sim, 0, 0, 0, 1.0, 1.0, yaw)
    act = np.array([[[0.5], [0.0], [0.0]]], np.float32); av = np.ones((1, 1), np.uint8)
    for t in range(5):
        oracle.step(log, sim, t, oracle.DYN_DELTA_LOCAL, act, av)
    assert sim["x"][0, 5, 0] == pytest.approx(1.0 + 2.5 * math.cos(yaw), abs=1e-6)
    assert sim["y"][0, 5, 0] == pytest.approx(1.0 + 2.5 * math.sin(yaw), abs=1e-6)


# P5 / D8 / D9
def test_playback_and_validity_rules():
    import wm_scenarios as ws
    cfg = ws.make_config(1)
    log = cfg["log"]
    sim = oracle.reset(log)
    B, T, A = log["x"].shape
    t = 10
    # rows >= history are cleared by reset (a0)
    assert sim["valid"][:, 11:].sum() == 0 and np.all(sim["x"][:, 11:] == 0)
    for k in log:
        assert np.array_equal(sim[k][:, :11], log[k][:, :11], equal_nan=True)
    av = np.zeros((B, A), np.uint8)
    oracle.step(log, sim, t, oracle.DYN_BICYCLE, np.ascontiguousarray(cfg["actions"][:, 0]), av)
    for k in log:   # all action_valid = 0 -> bit-equal to the log row (NaN poison included)
        assert np.array_equal(sim[k][:, t + 1], log[k][:, t + 1], equal_nan=True), k
    ld = oracle.log_divergence(log, sim, t + 1)
    assert np.all(ld["dist"] == 0)
    assert np.array_equal(ld["valid"], log["valid"][:, t + 1])
    # controlled agents: valid'=1, size carried; invalid-at-t agents with action_valid=1 -> log row
    av[:] = 1
    sim = oracle.reset(log)
    oracle.step(log, sim, t, oracle.DYN_BICYCLE, np.ascontiguousarray(cfg["actions"][:, 0]), av)
    was_valid = log["valid"][:, t] == 1
    assert np.all(sim["valid"][:, t + 1][was_valid] == 1)
    assert np.array_equal(sim["length"][:, t + 1][was_valid], log["length"][:, t][was_valid])
    assert np.array_equal(sim["width"][:, t + 1][was_valid], log["width"][:, t][was_valid])
    for k in log:
        assert np.array_equal(sim[k][:, t + 1][~was_valid], log[k][:, t + 1][~was_valid], equal_nan=True)
    assert not np.isnan(sim["x"][:, t + 1][was_valid]).any()


# P11
def test_log_divergence_3_4_5():
    log = mk_traj(1, 1, 3, valid=1); sim = mk_traj(1, 1, 3, valid=1)
    set_agent(log, 0, 0, 0, 100.0, -50.0); set_agent(sim, 0, 0, 0, 103.0, -46.0)
    set_agent(log, 0, 0, 1, 1.0, 1.0, valid=0); set_agent(sim, 0, 0, 1, 9.0, 9.0)
    set_agent(log, 0, 0, 2, 1.0, 1.0); set_agent(sim, 0, 0, 2, 9.0, 9.0, valid=0)
    out = oracle.log_divergence(log, sim, 0)
    assert out["dist"][0, 0] == pytest.approx(5.0, abs=1e-6)
    assert list(out["valid"][0]) == [1, 0, 0]
    assert out["dist"][0, 1] == 0 and out["dist"][0, 2] == 0


# Table 3 row "Expert / Delta": Log ADE 0.00: replaying the log's own inverse
# delta actions (L335: delta = s' - s, expressed in the body frame for DeltaLocal) reproduces
# the log, so every step's log divergence is ~0.
def test_expert_delta_replay_has_zero_log_divergence():
    import wm_scenarios as ws
    cfg = ws.make_config(1, poison_invalid=False)
    log = cfg["log"]
    B, T, A = log["x"].shape
    sim = oracle.reset(log)
    av = np.ascontiguousarray(log["valid"][:, 10])
    worst = 0.0
    for t in range(10, 40):
        x0, y0, th0 = (sim[k][:, t].astype(np.float64) for k in ("x", "y", "yaw"))
        dxw = log["x"][:, t + 1] - x0; dyw = log["y"][:, t + 1] - y0
        c, s = np.cos(th0), np.sin(th0)
        act = np.stack([c * dxw + s * dyw, -s * dxw + c * dyw, log["yaw"][:, t + 1] - th0], axis=1)
        oracle.step(log, sim, t, oracle.DYN_DELTA_LOCAL, np.ascontiguousarray(act.astype(np.float32)), av)
        ld = oracle.log_divergence(log, sim, t + 1)
        worst = max(worst, float(ld["dist"].max()))
    assert worst < 5e-5   # float32 action rounding only; "0.00" in the paper's two decimals
