"""Pins of the oracle's route-progress ratio (O11).  CPU only."""
import numpy as np

import oracle
import wm_scenarios as ws
from util import mk_traj, set_agent


def straight_path(B, A, P, spacing=1.0, valid=None):
    xs = (np.arange(P) * spacing).astype(np.float32)
    pa = dict(x=np.broadcast_to(xs, (B, A, P)).copy(), y=np.zeros((B, A, P), np.float32),
              arc_len=np.broadcast_to(xs, (B, A, P)).copy(), valid=np.ones((B, A, P), np.uint8))
    if valid is not None:
        pa["valid"][:] = valid
    return pa


def _scene(sim_xy, log_first=(2.0, 0.0), log_last=(22.0, 0.0), T=5):
    A = len(sim_xy)
    log = mk_traj(1, T, A); sim = mk_traj(1, T, A)
    for a, (x, y) in enumerate(sim_xy):
        set_agent(log, 0, 1, a, *log_first); set_agent(log, 0, T - 2, a, *log_last)     # rows 0 and T-1 invalid on purpose (D34)
        set_agent(sim, 0, 2, a, x, y)
    return log, sim


def test_straight_path_closed_form():
    # path along +x, 1 m spacing, arc length = x: d_p = 2, d_q = 22 -> ratio = (round(x) - 2) / 20
    log, sim = _scene([(12.3, 0.4), (2.0, -3.0), (22.2, 5.0), (30.1, 0.0), (-7.0, 1.0)])
    r = oracle.route_progress(log, sim, 2, straight_path(1, 5, 41))
    assert r["valid"].tolist() == [[1, 1, 1, 1, 1]]
    assert np.allclose(r["ratio"][0], [0.5, 0.0, 1.0, 1.4, -0.1], atol=1e-6)     # > 1 after the logged end (L96), < 0 before the start
    assert r["closest"][0, 0].tolist() == [12, 2, 22, 30, 0] and np.all(r["closest"][0, 1] == 2) and np.all(r["closest"][0, 2] == 22)


def test_ties_go_to_the_lower_index_and_invalid_points_are_ignored():
    log, sim = _scene([(12.5, 0.0), (12.5, 0.0)])
    pa = straight_path(1, 2, 41)
    pa["valid"][0, 1, 12] = 0; pa["x"][0, 1, 12] = np.nan                   # agent 1: point 12 is not part of the path
    r = oracle.route_progress(log, sim, 2, pa)
    assert r["closest"][0, 0].tolist() == [12, 13]                          # exact tie 12 / 13 -> 12 (D33); without 12 -> 13
    assert np.allclose(r["ratio"][0], [0.5, 0.55], atol=1e-6)


def test_validity_rules():
    log, sim = _scene([(5.0, 0.0)] * 5)
    pa = straight_path(1, 5, 41)
    sim["valid"][0, 2, 0] = 0                                                # sim invalid at t
    pa["valid"][0, 1, :] = 0                                                 # no path
    log["valid"][0, :, 2] = 0                                                # never logged
    log["x"][0, 3, 3] = 2.2                                                  # logged end next to the logged start: d_q == d_p (D35)
    r = oracle.route_progress(log, sim, 2, pa)
    assert r["valid"][0].tolist() == [0, 0, 0, 0, 1] and np.all(r["ratio"][0, :4] == 0)
    assert abs(r["ratio"][0, 4] - 0.15) < 1e-6


def test_circular_path_is_the_angle_fraction():
    # path = quarter circle of radius 20 sampled every degree, arc length = 20 * angle; the logged trajectory runs from 10 to 70 degrees
    P = 91
    ang = np.deg2rad(np.arange(P))
    pa = dict(x=(20 * np.cos(ang)).astype(np.float32)[None, None], y=(20 * np.sin(ang)).astype(np.float32)[None, None],
              arc_len=(20 * ang).astype(np.float32)[None, None], valid=np.ones((1, 1, P), np.uint8))
    log = mk_traj(1, 3, 1); sim = mk_traj(1, 3, 1)
    set_agent(log, 0, 0, 0, 20 * np.cos(np.deg2rad(10)), 20 * np.sin(np.deg2rad(10)))
    set_agent(log, 0, 2, 0, 20 * np.cos(np.deg2rad(70)), 20 * np.sin(np.deg2rad(70)))
    set_agent(sim, 0, 1, 0, 23 * np.cos(np.deg2rad(40.2)), 23 * np.sin(np.deg2rad(40.2)))     # 3 m outside the arc at 40.2 degrees
    r = oracle.route_progress(log, sim, 1, pa)
    assert r["closest"][0, :, 0].tolist() == [40, 10, 70] and abs(r["ratio"][0, 0] - 0.5) < 1e-5


def test_log_playback_progress_runs_from_0_to_1_on_generated_paths():
    cfg = ws.make_config(1, n_steps=4)
    log = cfg["log"]
    pa = ws.make_paths(log)
    B, T, A = log["x"].shape
    alive = (log["valid"].sum(axis=1) == T)                                 # agents logged for the whole episode
    moved = np.hypot(log["x"][:, -1] - log["x"][:, 0], log["y"][:, -1] - log["y"][:, 0]) > 1.0
    r0 = oracle.route_progress(log, log, 0, pa); r1 = oracle.route_progress(log, log, T - 1, pa); rm = oracle.route_progress(log, log, T // 2, pa)
    sel = alive & moved
    assert sel.sum() > 20
    assert np.all(r0["ratio"][sel] == 0) and np.all(r1["ratio"][sel] == 1)   # the log's own first / last position (L96)
    assert np.all((rm["ratio"][sel] > 0) & (rm["ratio"][sel] <= 1))          # = 1 for agents that have braked to a stop by then
    assert (rm["ratio"][sel] < 1).sum() > sel.sum() // 2


def test_offroute_hand_cases():
    """O12 (L98), thresholds as arguments (D36): max_dist = 5 m, margin = 1 m.  On-route path along +x
    (y = 0), off-route path parallel at y = 4."""
    pts = [(10.0, 1.0), (10.0, 2.4), (10.0, 2.6), (10.0, -5.5), (10.0, -4.5), (10.3, 0.0)]
    A = len(pts)
    sim = mk_traj(1, 1, A)
    for a, (x, y) in enumerate(pts):
        set_agent(sim, 0, 0, a, x, y)
    on = straight_path(1, A, 41)
    off = straight_path(1, A, 41); off["y"][:] = 4.0
    r = oracle.offroute(sim, 0, on, off, 5.0, 1.0)
    # (10,1): d_on 1, d_off 3 -> on route.  (10,2.4): 2.4 vs 1.6 + 1 = 2.6 -> on.  (10,2.6): 2.6 vs 1.4 + 1 = 2.4 -> OFF.
    # (10,-5.5): d_on 5.5 > 5 -> OFF.  (10,-4.5): 4.5 -> on.  (10.3, 0): nearest point (10, 0): d_on 0.3 -> on.
    assert r["flag"][0].tolist() == [0, 0, 1, 1, 0, 0]
    assert np.allclose(r["dist_on"][0], [1.0, 2.4, 2.6, 5.5, 4.5, 0.3], atol=1e-6)
    # without off-route paths only the distance rule is left
    assert oracle.offroute(sim, 0, on, None, 5.0, 1.0)["flag"][0].tolist() == [0, 0, 0, 1, 0, 0]
    # invalid agents and agents without an on-route path are never flagged
    sim["valid"][0, 0, 3] = 0; on["valid"][0, 2, :] = 0
    r = oracle.offroute(sim, 0, on, off, 5.0, 1.0)
    assert r["flag"][0].tolist() == [0, 0, 0, 0, 0, 0] and r["dist_on"][0, 3] == 0 and r["dist_on"][0, 2] == 0


def test_route_progress_equals_the_float64_definition_outside_the_band():
    """The oracle takes the closest-point decision of D33 on the kernel's float32 key.  Pin: a float64 numpy
    restatement of L96 / D33-D35 (tests/defs_f64.py) gives the same ratio wherever the three closest points are
    decided by more than 1e-4 m."""
    import wm_scenarios as ws
    from defs_f64 import route_ratio_in_double
    cfg = ws.make_config(5, B=3, n_steps=1)
    log = cfg["log"]
    paths = ws.make_paths(log)
    paths["valid"][:, ::7, 5] = 0
    for t in (10, 47, 90):
        r = oracle.route_progress(log, log, t, paths)
        rd, dec = route_ratio_in_double(log, log, t, paths)
        chk = dec & (r["valid"] == 1)
        assert chk.sum() > 0.8 * (r["valid"] == 1).sum()
        assert np.all(np.abs(r["ratio"] - rd)[chk] <= 1e-6 * np.maximum(1.0, np.abs(rd[chk])))
