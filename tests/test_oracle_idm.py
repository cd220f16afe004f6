"""Pins of the oracle's IDM sim agent (O13, ref. [51] = Treiber, Hennecke, Helbing
2000).  What is pinned is what the published model fixes independently of this code: the free-road
ODE dv/dt = a_max (1 - (v/v0)^delta), the equilibrium gap s_e = (s0 + v T) / sqrt(1 - (v/v0)^delta), no
collision with a stopped obstacle, and the lead-selection / path-following readings D38-D41.  CPU only."""
import numpy as np

import oracle
from util import mk_traj, set_agent

DT = 0.1
PRM = oracle.IDM_DEFAULTS


def line_paths(B, A, P, spacing=0.5):
    xs = (np.arange(P) * spacing).astype(np.float32)
    return dict(x=np.broadcast_to(xs, (B, A, P)).copy(), y=np.zeros((B, A, P), np.float32),
                arc_len=np.broadcast_to(xs, (B, A, P)).copy(), valid=np.ones((B, A, P), np.uint8))


def run(sim, paths, idm, steps, t0=0):
    out = []
    for t in range(t0, t0 + steps):
        out.append(oracle.idm_step(sim, t, paths, idm))
    return out


def test_free_road_follows_the_published_ode():
    T = 402
    sim = mk_traj(1, T, 1)
    set_agent(sim, 0, 0, 0, 1.0, 0.0, 0.0, 0.0, 0.0)
    pa = line_paths(1, 1, 4000)
    res = run(sim, pa, np.ones((1, 1), np.uint8), 400)
    assert abs(res[0]["accel"][0, 0] - PRM["a_max"]) < 1e-6 and res[0]["lead"][0, 0] == -1      # standing start: a = a_max
    # independent integration of dv/dt = a_max (1 - (v/v0)^4) with a fine RK4 step
    f = lambda v: PRM["a_max"] * (1.0 - (v / PRM["v0"]) ** PRM["delta"])
    v, h = 0.0, 0.001
    for _ in range(int(round(40.0 / h))):
        k1 = f(v); k2 = f(v + 0.5 * h * k1); k3 = f(v + 0.5 * h * k2); k4 = f(v + h * k3)
        v += h * (k1 + 2 * k2 + 2 * k3 + k4) / 6
    v_sim = float(np.hypot(sim["vel_x"][0, 400, 0], sim["vel_y"][0, 400, 0]))
    assert abs(v_sim - v) < 0.05, (v_sim, v)                      # explicit Euler at 0.1 s against the exact solution
    assert 25.0 < v_sim < PRM["v0"]
    # it stays on its path, heading along it, and moves by the trapezoid of its speeds
    assert np.all(np.abs(sim["y"][0, :401, 0]) < 1e-6) and np.all(np.abs(sim["yaw"][0, 1:401, 0]) < 1e-6)
    x = sim["x"][0, :401, 0].astype(np.float64); sp = np.hypot(sim["vel_x"][0, :401, 0], sim["vel_y"][0, :401, 0]).astype(np.float64)
    assert np.allclose(np.diff(x), 0.5 * (sp[:-1] + sp[1:]) * DT, atol=2e-4)
    # at the desired speed the free-road acceleration vanishes
    sim2 = mk_traj(1, 2, 1); set_agent(sim2, 0, 0, 0, 1.0, 0.0, 0.0, PRM["v0"], 0.0)
    assert abs(oracle.idm_step(sim2, 0, pa, np.ones((1, 1), np.uint8))["accel"][0, 0]) < 1e-6


def test_equilibrium_gap_of_the_published_model_is_a_fixed_point():
    v = 10.0
    s_e = (PRM["s0"] + v * PRM["T"]) / np.sqrt(1.0 - (v / PRM["v0"]) ** PRM["delta"])       # ref. [51], equilibrium
    L = 4.0
    sim = mk_traj(1, 3, 2)
    set_agent(sim, 0, 0, 0, 50.0, 0.0, 0.0, v, 0.0, length=L)                               # follower
    set_agent(sim, 0, 0, 1, 50.0 + s_e + L, 0.0, 0.0, v, 0.0, length=L)                     # leader, bumper gap s_e
    pa = line_paths(1, 2, 1000)
    r = oracle.idm_step(sim, 0, pa, np.array([[1, 0]], np.uint8))
    assert r["lead"][0, 0] == 1 and abs(r["accel"][0, 0]) < 2e-4
    assert abs(np.hypot(sim["vel_x"][0, 1, 0], sim["vel_y"][0, 1, 0]) - v) < 1e-4
    assert sim["valid"][0, 1, 1] == 0                                                       # D41: the uncontrolled slot is not written
    # closer than the equilibrium gap it brakes, farther it accelerates
    for dg, sign in ((-3.0, -1), (+3.0, +1)):
        s2 = mk_traj(1, 2, 2)
        set_agent(s2, 0, 0, 0, 50.0, 0.0, 0.0, v, 0.0, length=L); set_agent(s2, 0, 0, 1, 50.0 + s_e + dg + L, 0.0, 0.0, v, 0.0, length=L)
        assert np.sign(oracle.idm_step(s2, 0, pa, np.array([[1, 0]], np.uint8))["accel"][0, 0]) == sign


def test_stops_behind_a_standing_obstacle_without_touching_it():
    T = 402
    sim = mk_traj(1, T, 2)
    set_agent(sim, 0, 0, 0, 5.0, 0.0, 0.0, 12.0, 0.0, length=4.5)
    for t in range(T):
        set_agent(sim, 0, t, 1, 120.0, 0.3, 0.0, 0.0, 0.0, length=5.0)                      # parked on the path (playback rows)
    pa = line_paths(1, 2, 1000)
    run(sim, pa, np.array([[1, 0]], np.uint8), 400)
    x = sim["x"][0, :401, 0]
    gap = 120.0 - x - 0.5 * (4.5 + 5.0)
    assert gap.min() > 0.5                                        # "to avoid collisions" (L110): never touches
    assert np.hypot(sim["vel_x"][0, 400, 0], sim["vel_y"][0, 400, 0]) < 0.05 and abs(gap[400] - PRM["s0"]) < 0.5
    assert np.all(np.diff(x) >= -1e-6)                            # never drives backwards


def test_lead_selection_rules():
    sim = mk_traj(1, 2, 6)
    set_agent(sim, 0, 0, 0, 50.0, 0.0, 0.0, 10.0, 0.0, length=4.0, width=2.0)               # the IDM agent
    set_agent(sim, 0, 0, 1, 30.0, 0.0, 0.0, 10.0, 0.0)                                      # behind: ignored
    set_agent(sim, 0, 0, 2, 70.0, 2.6, 0.0, 10.0, 0.0, width=2.0)                           # beside the path (2.6 > (2+2)/2): ignored
    set_agent(sim, 0, 0, 3, 90.0, 0.5, 0.0, 3.0, 0.0, length=4.0)                           # ahead, far
    set_agent(sim, 0, 0, 4, 75.0, -1.5, 0.0, 5.0, 0.0, length=4.0, width=2.0)               # ahead, nearer, lateral 1.5 <= 2: THE lead
    set_agent(sim, 0, 0, 5, 60.0, 0.0, 0.0, 0.0, 0.0, valid=0)                              # invalid: ignored
    pa = line_paths(1, 6, 1000)
    idm = np.zeros((1, 6), np.uint8); idm[0, 0] = 1
    r = oracle.idm_step(sim, 0, pa, idm)
    assert r["lead"][0, 0] == 4
    sim["valid"][0, 0, 4] = 0
    assert oracle.idm_step(sim, 0, pa, idm)["lead"][0, 0] == 3
    sim["valid"][0, 0, 3] = 0
    assert oracle.idm_step(sim, 0, pa, idm)["lead"][0, 0] == -1
    # an agent without a path, or invalid at t, is not moved
    pa["valid"][0, 0, :] = 0; sim["valid"][0, 1, 0] = 0
    oracle.idm_step(sim, 0, pa, idm)
    assert sim["valid"][0, 1, 0] == 0


def test_follows_a_curved_path_and_stops_at_its_end():
    P = 181
    ang = np.deg2rad(np.arange(P) * 0.5)                           # quarter circle of radius 40, 0.349 m spacing
    pa = dict(x=(40 * np.cos(ang)).astype(np.float32)[None, None], y=(40 * np.sin(ang)).astype(np.float32)[None, None],
              arc_len=(40 * ang).astype(np.float32)[None, None], valid=np.ones((1, 1, P), np.uint8))
    T = 202
    sim = mk_traj(1, T, 1)
    set_agent(sim, 0, 0, 0, 40.0, 0.0, np.pi / 2, 0.0, 8.0)
    run(sim, pa, np.ones((1, 1), np.uint8), 200)
    r = np.hypot(sim["x"][0, :201, 0], sim["y"][0, :201, 0])
    assert np.all(r <= 40.0 + 1e-4) and np.all(r >= 40.0 * np.cos(np.deg2rad(0.25)) - 1e-4)     # on the chords of the polyline
    th = np.arctan2(sim["y"][0, 1:50, 0], sim["x"][0, 1:50, 0])
    assert np.all(np.abs(np.angle(np.exp(1j * (sim["yaw"][0, 1:50, 0] - (th + np.pi / 2))))) < np.deg2rad(0.5))   # tangent heading
    # 20 s at >= 8 m/s is more than the 62.8 m of path: it ends on the last point
    assert abs(sim["x"][0, 200, 0] - pa["x"][0, 0, -1]) < 1e-5 and abs(sim["y"][0, 200, 0] - pa["y"][0, 0, -1]) < 1e-5


def test_lead_choice_equals_the_float64_definition_outside_the_band():
    """The oracle takes the lead decision of D39 in float32, operation for operation as the kernel does.  Pin: a
    float64 numpy restatement of the definition (tests/defs_f64.py) picks the same lead wherever every comparison
    behind the choice is clear by more than 1e-4 m; that is nearly everywhere on the config-5 traffic."""
    import wm_scenarios as ws
    from defs_f64 import idm_lead_in_double
    cfg = ws.make_config(5, B=3, n_steps=1)
    log = cfg["log"]
    B, T, A = log["x"].shape
    paths = ws.make_paths(log)
    idm = np.ones((B, A), np.uint8); idm[:, ::6] = 0
    n_ctl = n_dec = n_lead = 0
    for t in (10, 33):
        sim = {k: v.copy() for k, v in log.items()}
        r = oracle.idm_step(sim, t, paths, idm)
        ld, dec = idm_lead_in_double(log, t, paths, idm)
        ctl = (idm == 1) & (log["valid"][:, t] == 1)
        assert np.array_equal(r["lead"][dec & ctl], ld[dec & ctl])
        n_ctl += int(ctl.sum()); n_dec += int((dec & ctl).sum()); n_lead += int(((ld >= 0) & dec & ctl).sum())
    assert n_dec > 0.9 * n_ctl and n_lead > 50
