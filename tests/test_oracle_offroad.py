"""Pins for the oracle's offroad signed distance (O4, readings D14-D20)."""
import math

import numpy as np
import pytest

import oracle
from util import boxes_traj, mk_roadgraph, rigid

EPS_BOX = (1e-3, 1e-3)   # a tiny box: its 4 corners are (almost) a single query point


def _point_query(rg, pts):
    """signed distance of near-point boxes centred at pts (yaw 0, 1 mm square)."""
    tr = boxes_traj([(x, y, 0.0, *EPS_BOX) for x, y in pts])
    return oracle.offroad(tr, 0, rg)


# P9a: single straight edge along +x from (0,0) to (10,0): left (y>0) is on-road (negative).
def test_straight_edge_closed_form():
    line = np.stack([np.arange(0, 10.5, 0.5), np.zeros(21)], 1)
    rg = mk_roadgraph([line])
    pts = [(2.0, 3.0), (7.3, -1.25), (5.0, 0.75), (-3.0, 4.0), (13.0, -4.0), (12.0, 0.5)]
    out = _point_query(rg, pts)
    exp = [-3.0, 1.25, -0.75, -5.0, 5.0, -math.hypot(2.0, 0.5)]
    # corner values differ from the centre value by at most the 1 mm box half-diagonal
    for a, e in enumerate(exp):
        assert out["signed_dist"][0, a] == pytest.approx(e, abs=1.5e-3), (a, e)
        assert out["flag"][0, a] == (1 if e > 0 else 0)


def test_corner_values_and_max_rule_D18():
    # vehicle 4 x 2 at (5, 0.5), yaw 0, over the straight edge y=0 (on-road side y>0):
    # corners FL(7,1.5) FR(7,-0.5) RR(3,-0.5) RL(3,1.5) -> sd = -1.5, +0.5, +0.5, -1.5
    line = np.stack([np.arange(0, 10.5, 0.5), np.zeros(21)], 1)
    rg = mk_roadgraph([line])
    out = oracle.offroad(boxes_traj([(5.0, 0.5, 0.0, 4.0, 2.0)]), 0, rg)
    assert np.allclose(out["corner_dist"][0, :, 0], [-1.5, 0.5, 0.5, -1.5], atol=1e-6)
    assert out["signed_dist"][0, 0] == pytest.approx(0.5, abs=1e-6) and out["flag"][0, 0] == 1
    # yaw = 90 deg: FL(4.0,2.5) FR(6.0,2.5) RR(6.0,-1.5) RL(4.0,-1.5)
    out = oracle.offroad(boxes_traj([(5.0, 0.5, math.pi / 2, 4.0, 2.0)]), 0, rg)
    assert np.allclose(out["corner_dist"][0, :, 0], [-2.5, -2.5, 1.5, 1.5], atol=1e-5)


# P9b: CCW circular arc of radius rho (left = inside): sd = r - rho up to the sagitta
# rho(1-cos(ds/2rho)) ~ ds^2/(8 rho).
def test_ccw_circle_closed_form():
    rho, ds = 20.0, 0.5
    n = int(round(2 * math.pi * rho / ds))
    ang = np.arange(n + 1) * (2 * math.pi / n)
    circ = np.stack([rho * np.cos(ang), rho * np.sin(ang)], 1)
    rg = mk_roadgraph([circ])
    sag = rho * (1 - math.cos(math.pi / n))
    assert sag == pytest.approx(ds * ds / (8 * rho), rel=0.01)
    rs = [5.0, 15.0, 19.5, 20.5, 27.0]
    th = [0.3, 2.0, 4.0, 5.5, 1.234]
    out = _point_query(rg, [(r * math.cos(t), r * math.sin(t)) for r, t in zip(rs, th)])
    for a, r in enumerate(rs):
        v = out["signed_dist"][0, a]
        assert r - rho - 1.5e-3 <= v <= r - rho + sag + 1.5e-3, (r, v)
        assert out["flag"][0, a] == (1 if r > rho else 0)


# P9c: reversing a polyline's point order flips every sign and keeps every magnitude.
def test_reversal_flips_sign():
    import wm_scenarios as ws
    cfg = ws.make_config(1, poison_invalid=False)
    rg = cfg["roadgraph"]; tr = cfg["log"]
    out = oracle.offroad(tr, 10, rg)
    rev = {k: np.ascontiguousarray(v[:, ::-1]) for k, v in rg.items()}
    rev["dir_x"] = -rev["dir_x"]; rev["dir_y"] = -rev["dir_y"]
    out2 = oracle.offroad(tr, 10, rev)
    ok = (out["ambig"] == 0) & (out2["ambig"] == 0) & (tr["valid"][:, 10][:, None, :] == 1)
    assert ok.mean() > 0.5
    assert np.allclose(out2["corner_dist"][ok], -out["corner_dist"][ok], atol=1e-6)


# P10a: rigid-transform invariance of all signed distances (outside the band)
def test_rigid_invariance():
    import wm_scenarios as ws
    cfg = ws.make_config(1, poison_invalid=False)
    out = oracle.offroad(cfg["log"], 10, cfg["roadgraph"])
    tr2, rg2 = rigid(cfg["log"], cfg["roadgraph"], -1.2, 33.0, 71.0)
    out2 = oracle.offroad(tr2, 10, rg2)
    ok = (out["ambig"] == 0) & (out2["ambig"] == 0)
    assert np.allclose(out2["corner_dist"][ok], out["corner_dist"][ok], atol=3e-4)
    okf = ok.all(axis=1)
    assert np.array_equal(out2["flag"][okf], out["flag"][okf])


# P10b: |sd| equals an independently coded min point-to-segment distance (numpy, vectorised,
# via the projection-free formula: distance to the line if the foot is inside, else to the
# nearer endpoint).
def test_abs_equals_independent_point_segment_distance():
    import wm_scenarios as ws
    cfg = ws.make_config(1, poison_invalid=False)
    rg, tr = cfg["roadgraph"], cfg["log"]
    out = oracle.offroad(tr, 10, rg)
    b = 1
    x, y, ty, idd = (rg[k][b].astype(np.float64) for k in ("x", "y", "type", "id"))
    m = (ty[:-1] == 2) & (ty[1:] == 2) & (idd[:-1] == idd[1:])
    p0 = np.stack([x[:-1], y[:-1]], 1)[m]; p1 = np.stack([x[1:], y[1:]], 1)[m]
    assert len(p0) == oracle.count_segments(rg, b)
    e = p1 - p0; L = np.linalg.norm(e, axis=1); u = e / L[:, None]
    for a in range(tr["x"].shape[2]):
        if not tr["valid"][b, 10, a]:
            continue
        cx, cy, th, ln, wd = (float(tr[k][b, 10, a]) for k in ("x", "y", "yaw", "length", "width"))
        f = np.array([math.cos(th), math.sin(th)]); s = np.array([-f[1], f[0]])
        for k, (sl, sw) in enumerate(((1, 1), (1, -1), (-1, -1), (-1, 1))):
            q = np.array([cx, cy]) + sl * ln / 2 * f + sw * wd / 2 * s
            w = q - p0
            al = (w * u).sum(1)
            perp = np.abs(w[:, 0] * u[:, 1] - w[:, 1] * u[:, 0])
            d = np.where(al < 0, np.linalg.norm(w, axis=1), np.where(al > L, np.linalg.norm(q - p1, axis=1), perp))
            assert abs(out["corner_dist"][b, k, a]) == pytest.approx(d.min(), abs=1e-5)


# P10c: lane pair of edges 3.5 m apart (orientation rule: carriageway on the left of both)
def test_lane_pair_flags():
    xs = np.arange(0, 40.5, 0.5)
    right_edge = np.stack([xs, np.full_like(xs, -1.75)], 1)            # runs +x: left is +y
    left_edge = np.stack([xs[::-1], np.full_like(xs, 1.75)], 1)        # runs -x: left is -y
    rg = mk_roadgraph([right_edge, left_edge])
    W = 2.0
    shift = (3.5 - W) / 2
    boxes = [(20.0, 0.0, 0.0, 4.5, W), (20.0, shift + 0.01, 0.0, 4.5, W), (20.0, -(shift + 0.01), 0.0, 4.5, W),
             (20.0, shift - 0.01, 0.0, 4.5, W)]
    out = oracle.offroad(boxes_traj(boxes), 0, rg)
    assert list(out["flag"][0]) == [0, 1, 1, 0]
    assert out["signed_dist"][0, 0] == pytest.approx(-shift, abs=1e-6)
    assert out["signed_dist"][0, 1] == pytest.approx(0.01, abs=1e-6)


# P10d: lane-typed and invalid points never change the result; splitting a polyline id at a
# vertex only removes that one segment.
def test_lane_and_invalid_points_ignored_and_id_split():
    xs = np.arange(0, 20.5, 0.5)
    edge = np.stack([xs, np.zeros_like(xs)], 1)
    lane = np.stack([xs, np.full_like(xs, 1.0)], 1)       # closer to the query than the edge
    rg_a = mk_roadgraph([edge])
    rg_b = mk_roadgraph([lane, edge, lane + [0, 0.2]], types=[1, 2, 1])
    rg_c = mk_roadgraph([edge, lane])                      # 2nd polyline road-edge typed but invalid
    rg_c["valid"][:, len(xs):] = 0
    boxes = [(5.0, 2.0, 0.3, 4.0, 2.0), (12.0, -3.0, 2.0, 4.0, 2.0)]
    ref = oracle.offroad(boxes_traj(boxes), 0, rg_a)
    for rg in (rg_b, rg_c):
        o = oracle.offroad(boxes_traj(boxes), 0, rg)
        assert np.array_equal(o["corner_dist"], ref["corner_dist"])
    assert oracle.count_segments(rg_a, 0) == len(xs) - 1
    rg_d = mk_roadgraph([edge])
    rg_d["id"][:, 21:] = 7                                  # split between points 20 and 21
    assert oracle.count_segments(rg_d, 0) == len(xs) - 2
    # a query right above the removed segment now snaps to the neighbouring vertices
    o = _point_query(rg_d, [(10.25, 1.0)])
    assert abs(o["signed_dist"][0, 0]) == pytest.approx(math.hypot(0.25, 1.0), abs=2e-3)


def test_isolated_point_uses_stored_dir_and_empty_roadgraph_D16_D20():
    rg = mk_roadgraph([np.array([[0.0, 0.0]])])
    rg["dir_x"][:] = 0.0; rg["dir_y"][:] = 1.0            # edge runs +y: left is -x
    assert oracle.count_segments(rg, 0) == 1
    o = _point_query(rg, [(-3.0, 4.0), (3.0, 4.0)])
    assert o["signed_dist"][0, 0] == pytest.approx(-5.0, abs=2e-3)
    assert o["signed_dist"][0, 1] == pytest.approx(5.0, abs=2e-3)
    rg["type"][:] = 1                                      # no road edge at all
    o = oracle.offroad(boxes_traj([(1.0, 1.0, 0.0, 4.0, 2.0)]), 0, rg)
    assert o["signed_dist"][0, 0] == -np.finfo(np.float32).max and o["flag"][0, 0] == 0


def test_tie_goes_to_lower_index_D17():
    # Query exactly above the shared vertex of a > 90 degree turn: both neighbours are at the
    # same distance with opposite signs; the lower-index segment decides.
    poly = np.array([[-4.0, 0.0], [0.0, 0.0], [-3.0, 3.0]])   # turns by 135 degrees at the origin
    rg = mk_roadgraph([poly])
    tr = boxes_traj([(2.0, 1.0, 0.0, 1e-6, 1e-6)])
    o = oracle.offroad(tr, 0, rg)
    # segment 0 runs +x: the point (2,1) is on its left (-> negative); segment 1 would say positive
    assert o["win_seg"][0, 0, 0] == 0
    assert o["corner_dist"][0, 0, 0] == pytest.approx(-math.hypot(2, 1), abs=1e-5)
    assert o["ambig"][0, 0, 0] == 1                         # and it is flagged ambiguous (P15)


def test_invalid_agents_output_zero_D10():
    rg = mk_roadgraph([np.array([[0.0, 0.0], [5.0, 0.0]])])
    tr = boxes_traj([(1.0, 1.0, 0.0, 4.0, 2.0), (2.0, -1.0, 0.0, 4.0, 2.0)])
    tr["valid"][0, 0, 1] = 0
    for k in ("x", "y", "yaw", "length", "width"):
        tr[k][0, 0, 1] = np.nan
    o = oracle.offroad(tr, 0, rg)
    assert o["signed_dist"][0, 1] == 0 and o["flag"][0, 1] == 0 and np.all(o["corner_dist"][0, :, 1] == 0)
