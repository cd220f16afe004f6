"""Pins of the oracle's expert inverse (O9) and kinematic-infeasibility metric (O10).

PAPER.md L335 (delta inverse), L352-L359 (Eq. 3), L104 (limits 6 m/s^2, 0.3 1/m), L198 ("By
construction the bicycle action space does not violate the kinematic metric"), Table 3
(Expert / Delta: Log ADE 0.00).  CPU only.
"""
import os

import numpy as np
import pytest

import oracle
from util import mk_traj, set_agent

DT = 0.1
GOLD = os.path.join(os.path.dirname(__file__), "golden", "kinematic_hand_cases.txt")


def _cases():
    out = []
    for line in open(GOLD):
        line = line.split("#")[0].split()
        if len(line) == 8:
            out.append([float(v) for v in line])
    return out


def test_golden_hand_cases():
    cases = _cases()
    assert len(cases) >= 11
    tr = mk_traj(1, 2, len(cases))
    for a, (yaw, vx, vy, vx1, vy1, *_r) in enumerate(cases):
        set_agent(tr, 0, 0, a, 0, 0, yaw, vx, vy)
        set_agent(tr, 0, 1, a, 0, 0, yaw, vx1, vy1)
    k = oracle.kinematic(tr, 1)
    e = oracle.expert_actions(tr, 0, 1, oracle.DYN_BICYCLE)
    for a, (yaw, vx, vy, vx1, vy1, acc, kap, flag) in enumerate(cases):
        assert k["valid"][0, 0, a] == 1
        assert abs(k["accel"][0, 0, a] - acc) < 2e-4, (a, k["accel"][0, 0, a], acc)
        want_k = kap
        assert abs(k["curvature"][0, 0, a] - want_k) < 2e-4 * max(1.0, abs(want_k)), (a, k["curvature"][0, 0, a], want_k)
        if abs(abs(want_k) - 0.3) > 1e-3 and abs(abs(acc) - 6.0) > 1e-3:      # the kappa = 0.3 row sits on the boundary
            assert k["flag"][0, 0, a] == int(flag), a
        # the expert actor IS the same inverse (L204)
        assert e["action"][0, 0, 0, a] == k["accel"][0, 0, a] and e["action"][0, 0, 1, a] == k["curvature"][0, 0, a]


def test_bicycle_inverse_round_trip_and_feasible_by_construction():
    """P3 + L198: step (Eq. 2) then inverse (Eq. 3) returns the action; actions inside the limits
    are never flagged."""
    rng = np.random.default_rng(5)
    A = 256
    log = mk_traj(1, 3, A, valid=1)
    sim = mk_traj(1, 3, A, valid=1)
    yaw = rng.uniform(-7.0, 7.0, A)                  # yaw is not wrapped in step (D5): beyond +-pi on purpose
    spd = rng.uniform(0.5, 15.0, A)
    for a in range(A):
        set_agent(sim, 0, 0, a, rng.uniform(-50, 50), rng.uniform(-50, 50), yaw[a], spd[a] * np.cos(yaw[a]), spd[a] * np.sin(yaw[a]))
    act = np.zeros((1, 2, A), np.float32)
    act[0, 0] = rng.uniform(-5.9, 5.9, A); act[0, 1] = rng.uniform(-0.29, 0.29, A)
    oracle.step(log, sim, 0, oracle.DYN_BICYCLE, act, np.ones((1, A), np.uint8))
    e = oracle.expert_actions(sim, 0, 1, oracle.DYN_BICYCLE)
    den = e["kden"][0, 0]
    assert np.all(e["valid"] == 1) and np.all(den > 0)
    assert np.abs(e["action"][0, 0, 0] - act[0, 0]).max() < 1e-3                 # float32 state: dv ~ 1e-6 / dt
    assert np.all(np.abs(e["action"][0, 0, 1] - act[0, 1]) < 2e-6 / den + 1e-5)  # heading ulp / distance travelled
    k = oracle.kinematic(sim, 1)
    assert k["flag"].sum() == 0                                                 # L198
    # and an action outside the limits, applied unclipped, IS flagged
    sim2 = {q: v.copy() for q, v in sim.items()}
    act2 = act.copy(); act2[0, 0, : A // 2] = 7.5; act2[0, 1, A // 2:] = 0.4; act2[0, 0, A // 2:] = 0.0
    oracle.step(log, sim2, 0, oracle.DYN_BICYCLE, act2, np.ones((1, A), np.uint8), max_accel=0.0, max_curvature=0.0)
    assert oracle.kinematic(sim2, 1)["flag"].sum() == A


def test_delta_inverse_hand_case_and_body_frame():
    tr = mk_traj(1, 2, 3, valid=1)
    set_agent(tr, 0, 0, 0, 1.0, 2.0, np.pi / 2, 0, 0); set_agent(tr, 0, 1, 0, 1.0, 3.0, np.pi / 2 + 0.25, 0, 0)   # moved 1 m along its heading
    set_agent(tr, 0, 0, 1, 0.0, 0.0, 0.0, 0, 0); set_agent(tr, 0, 1, 1, 0.3, -0.4, -0.1, 0, 0)                  # yaw 0: Eq. 1 literally (L335)
    set_agent(tr, 0, 0, 2, 5.0, 5.0, np.pi, 0, 0); set_agent(tr, 0, 1, 2, 4.0, 5.5, np.pi, 0, 0)                # facing -x: forward 1, left -0.5
    e = oracle.expert_actions(tr, 0, 1, oracle.DYN_DELTA_LOCAL)["action"][0, 0]
    assert np.allclose(e[:, 0], [1.0, 0.0, 0.25], atol=1e-6)
    assert np.allclose(e[:, 1], [0.3, -0.4, -0.1], atol=1e-6)
    assert np.allclose(e[:, 2], [1.0, -0.5, 0.0], atol=1e-6)


def test_expert_delta_replay_has_zero_log_divergence():
    """Table 3: Expert / Delta has Log ADE 0.00 - replaying the inverse-delta actions of the
    log reproduces the log."""
    import wm_scenarios as ws
    cfg = ws.make_config(1, n_steps=80)
    log, rg = cfg["log"], cfg["roadgraph"]
    e = oracle.expert_actions(log, cfg["t0"], 80, oracle.DYN_DELTA_LOCAL)
    sim = oracle.reset(log)
    out = oracle.rollout(log, sim, rg, cfg["t0"], 80, oracle.DYN_DELTA_LOCAL, e["action"], e["valid"])
    assert out["ade"].max() < 5e-3 and round(float(out["ade"].max()), 2) == 0.0
    v = (sim["valid"] == 1) & (log["valid"] == 1)
    assert np.abs(sim["yaw"][v] - log["yaw"][v]).max() < 1e-4


def test_validity_and_poison():
    tr = mk_traj(1, 3, 4, valid=1)
    for t in range(3):
        for a in range(4):
            set_agent(tr, 0, t, a, t * 1.0, 0, 0, 10, 0)
    tr["valid"][0, 1, 1] = 0; tr["vel_x"][0, 1, 1] = np.nan
    tr["valid"][0, 2, 2] = 0; tr["x"][0, 2, 2] = np.nan; tr["vel_y"][0, 2, 2] = np.nan
    k = oracle.kinematic(tr, 1, 2)
    assert k["valid"][0, :, 1].tolist() == [0, 0] and k["valid"][0, :, 2].tolist() == [1, 0] and k["valid"][0, :, 0].tolist() == [1, 1]
    assert np.isfinite(k["accel"]).all() and np.isfinite(k["curvature"]).all() and k["flag"].sum() == 0
    for dyn in (oracle.DYN_BICYCLE, oracle.DYN_DELTA_LOCAL):
        e = oracle.expert_actions(tr, 0, 2, dyn)
        assert np.array_equal(e["valid"], k["valid"]) and np.isfinite(e["action"]).all()
        assert np.all(e["action"][0, :, :, 1] == 0) and np.all(e["action"][0, 1, :, 2] == 0)


def test_rigid_invariance_of_the_bicycle_inverse():
    rng = np.random.default_rng(11)
    A = 64
    tr = mk_traj(1, 2, A, valid=1)
    for t in range(2):
        for a in range(A):
            th = rng.uniform(-3, 3); v = rng.uniform(0.2, 12)
            set_agent(tr, 0, t, a, rng.uniform(-20, 20), rng.uniform(-20, 20), th, v * np.cos(th + 0.01 * t), v * np.sin(th + 0.01 * t))
    from util import rigid
    tr2, _ = rigid(tr, None, 0.7, 30.0, -12.0)
    k1, k2 = oracle.kinematic(tr, 1), oracle.kinematic(tr2, 1)
    assert np.abs(k1["accel"] - k2["accel"]).max() < 1e-3
    assert np.all(np.abs(k1["curvature"] - k2["curvature"]) < 4e-6 / k1["kden"] + 1e-5)


def test_delta_global_is_eq1_literally():
    """Eq. 1 (L324-L333): x' = x + dx, y' = y + dy, yaw' = yaw + dyaw, v' = (p' - p)/dt, whatever
    the yaw; its inverse (L335) is the plain difference."""
    rng = np.random.default_rng(3)
    A = 32
    log = mk_traj(1, 2, A, valid=1); sim = mk_traj(1, 2, A, valid=1)
    st = rng.uniform(-30, 30, (A, 3))
    for a in range(A):
        set_agent(sim, 0, 0, a, st[a, 0], st[a, 1], st[a, 2] * 0.2, 1.0, 2.0)
    act = np.zeros((1, 3, A), np.float32)
    act[0, 0] = rng.uniform(-0.5, 0.5, A); act[0, 1] = rng.uniform(-0.5, 0.5, A); act[0, 2] = rng.uniform(-0.1, 0.1, A)
    x0, y0, th0 = sim["x"][0, 0].astype(np.float64), sim["y"][0, 0].astype(np.float64), sim["yaw"][0, 0].astype(np.float64)
    oracle.step(log, sim, 0, oracle.DYN_DELTA_GLOBAL, act, np.ones((1, A), np.uint8))
    assert np.allclose(sim["x"][0, 1], x0 + act[0, 0], atol=4e-6) and np.allclose(sim["y"][0, 1], y0 + act[0, 1], atol=4e-6)
    assert np.allclose(sim["yaw"][0, 1], th0 + act[0, 2], atol=1e-6)
    assert np.allclose(sim["vel_x"][0, 1], (sim["x"][0, 1].astype(np.float64) - x0) / DT, atol=1e-5)
    assert np.allclose(sim["vel_y"][0, 1], (sim["y"][0, 1].astype(np.float64) - y0) / DT, atol=1e-5)
    e = oracle.expert_actions(sim, 0, 1, oracle.DYN_DELTA_GLOBAL)["action"][0, 0]
    assert np.allclose(e, act[0], atol=4e-6)
    # and with yaw = 0 the local and the global model coincide (D2)
    sim0 = mk_traj(1, 2, A, valid=1); sim1 = mk_traj(1, 2, A, valid=1)
    for a in range(A):
        set_agent(sim0, 0, 0, a, st[a, 0], st[a, 1], 0.0, 1.0, 2.0); set_agent(sim1, 0, 0, a, st[a, 0], st[a, 1], 0.0, 1.0, 2.0)
    oracle.step(log, sim0, 0, oracle.DYN_DELTA_GLOBAL, act, np.ones((1, A), np.uint8))
    oracle.step(log, sim1, 0, oracle.DYN_DELTA_LOCAL, act, np.ones((1, A), np.uint8))
    for k in ("x", "y", "yaw", "vel_x", "vel_y"):
        assert np.array_equal(sim0[k], sim1[k]), k
