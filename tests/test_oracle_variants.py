"""Pins for the SURVEY 8(f)(4) variants of the oracle: backward pass of the dynamics (O14, PAPER.md
L252), discretised action spaces (O15, L204) and the sorted-by-distance top-k order (O7 / D44).

Expected values come from what the mathematics fixes independently of the code under test: central
finite differences of the (separately pinned) forward step, the kappa = 0 closed form of Eq. 2,
hand-worked grids, numpy's sort.
"""
import math

import numpy as np
import pytest

import oracle
from util import mk_traj, set_agent, mk_roadgraph

DT = 0.1


# ---------------------------------------------------------------------------------------
# O14 backward pass
# ---------------------------------------------------------------------------------------
def _forward(dyn, s0, acts, av=None, clip=(0.0, 0.0)):
    """n oracle steps of one agent from state s0 = (x, y, yaw, vx, vy); returns rows [n+1][5] (float64 of the float32 rows)."""
    n = acts.shape[0]
    T = n + 1
    log = mk_traj(1, T, 1, valid=1)
    for t in range(T):
        set_agent(log, 0, t, 0, 100.0 + t, -50.0, 0.3, 1.0, 2.0)
    sim = mk_traj(1, T, 1, valid=0)
    set_agent(sim, 0, 0, 0, *s0)
    for t in range(n):
        a = np.ascontiguousarray(acts[t].reshape(1, -1, 1), np.float32)
        v = np.ones((1, 1), np.uint8) if av is None else np.full((1, 1), av[t], np.uint8)
        oracle.step(log, sim, t, dyn, a, v, dt=DT, max_accel=clip[0], max_curvature=clip[1])
    rows = np.stack([sim[k][0, :, 0].astype(np.float64) for k in ("x", "y", "yaw", "vel_x", "vel_y")], axis=1)
    return rows, sim


def _vjp(dyn, sim, acts, g_rows, av=None, clip=(0.0, 0.0)):
    n = acts.shape[0]
    a = np.ascontiguousarray(acts.reshape(1, n, -1, 1), np.float32)
    v = np.ones((1, n, 1), np.uint8) if av is None else np.asarray(av, np.uint8).reshape(1, n, 1)
    g = np.ascontiguousarray(g_rows.reshape(1, n, 5, 1), np.float32)
    r = oracle.rollout_vjp(sim, 0, n, dyn, a, v, g, dt=DT, max_accel=clip[0], max_curvature=clip[1])
    return r["g_actions"][0, :, :, 0].astype(np.float64), r["g_state0"][0, :, 0].astype(np.float64)


@pytest.mark.parametrize("dyn,C", [(oracle.DYN_BICYCLE, 2), (oracle.DYN_DELTA_LOCAL, 3), (oracle.DYN_DELTA_GLOBAL, 3)])
def test_vjp_matches_central_differences_of_the_forward_step(dyn, C):
    """The loss L = sum_k w_k . row_k of a 6-step rollout: its gradient w.r.t. every action and the
    initial state equals (L(+eps) - L(-eps)) / 2 eps of the oracle's own forward step (pinned in
    test_oracle_dynamics.py).  States near the origin keep the float32 rounding of the rows small."""
    rng = np.random.default_rng(7 + dyn)
    n = 6
    s0 = np.array([0.3, -0.2, 0.4, 1.2 * math.cos(0.4), 1.2 * math.sin(0.4)])
    if dyn == oracle.DYN_BICYCLE:
        acts = np.stack([rng.uniform(-2, 2, n), rng.uniform(-0.2, 0.2, n)], axis=1)
    else:
        acts = np.stack([rng.uniform(-0.3, 0.3, n), rng.uniform(-0.3, 0.3, n), rng.uniform(-0.1, 0.1, n)], axis=1)
    w = rng.uniform(-1, 1, (n, 5))
    rows, sim = _forward(dyn, s0, acts)
    ga, g0 = _vjp(dyn, sim, acts, w)

    def loss(s, a):
        r, _ = _forward(dyn, s, a)
        return float((w * r[1:]).sum())
    eps = 2e-2
    scale = max(1.0, np.abs(ga).max(), np.abs(g0).max())
    for k in range(n):
        for c in range(C):
            ap, am = acts.copy(), acts.copy()
            ap[k, c] += eps; am[k, c] -= eps
            fd = (loss(s0, ap) - loss(s0, am)) / (2 * eps)
            assert abs(fd - ga[k, c]) < 3e-3 * scale, (k, c, fd, ga[k, c])
    for j in range(5):
        sp, sm = s0.copy(), s0.copy()
        sp[j] += eps; sm[j] -= eps
        fd = (loss(sp, acts) - loss(sm, acts)) / (2 * eps)
        assert abs(fd - g0[j]) < 3e-3 * scale, (j, fd, g0[j])


def test_vjp_bicycle_straight_line_closed_form():
    """kappa = 0 (Eq. 2 is then the exact constant-acceleration integrator, L339-L350): with the loss
    x_n, d x_n / d a_k = cos(theta) dt^2 (1/2 + n - 1 - k), summing to cos(theta) (n dt)^2 / 2;
    d x_n / d v = n dt cos(theta) through (vx, vy) = v (cos, sin); d x_n / d x_0 = 1."""
    n, th, v0 = 20, 0.6, 4.0
    acts = np.zeros((n, 2)); acts[:, 0] = 1.5
    s0 = np.array([0.0, 0.0, th, v0 * math.cos(th), v0 * math.sin(th)])
    rows, sim = _forward(oracle.DYN_BICYCLE, s0, acts)
    w = np.zeros((n, 5)); w[-1, 0] = 1.0
    ga, g0 = _vjp(oracle.DYN_BICYCLE, sim, acts, w)
    for k in range(n):
        assert ga[k, 0] == pytest.approx(math.cos(th) * DT * DT * (0.5 + n - 1 - k), rel=1e-5)
    assert ga[:, 0].sum() == pytest.approx(math.cos(th) * (n * DT) ** 2 / 2, rel=1e-5)
    assert g0[0] == pytest.approx(1.0) and g0[1] == pytest.approx(0.0, abs=1e-7)
    # vx enters x' directly (dt) and through v = |(vx, vy)| for the later steps: (n-1) dt cos(th) * vx/v
    assert g0[3] == pytest.approx(DT + (n - 1) * DT * math.cos(th) * math.cos(th), rel=1e-5)
    assert g0[4] == pytest.approx((n - 1) * DT * math.cos(th) * math.sin(th), rel=1e-5)


def test_vjp_playback_and_clipping_pass_no_gradient():
    """D43: a playback step cuts the chain (its successor is the log's); an action beyond the clip
    limit has zero gradient while the state gradient still flows."""
    n = 4
    acts = np.array([[1.0, 0.05], [9.0, 0.5], [1.0, 0.05], [1.0, 0.05]])      # step 1 is clipped at (6, 0.3)
    s0 = np.array([0.0, 0.0, 0.2, 3.0 * math.cos(0.2), 3.0 * math.sin(0.2)])
    w = np.ones((n, 5))
    rows, sim = _forward(oracle.DYN_BICYCLE, s0, acts, clip=(6.0, 0.3))
    ga, g0 = _vjp(oracle.DYN_BICYCLE, sim, acts, w, clip=(6.0, 0.3))
    assert ga[1, 0] == 0.0 and ga[1, 1] == 0.0 and ga[0, 0] != 0.0 and np.abs(g0).sum() > 0
    av = [1, 1, 0, 1]                                                      # step 2 plays the log back
    rows, sim = _forward(oracle.DYN_BICYCLE, s0, acts, av=av, clip=(6.0, 0.3))
    ga, g0 = _vjp(oracle.DYN_BICYCLE, sim, acts, w, av=av, clip=(6.0, 0.3))
    assert np.all(ga[2] == 0.0) and ga[3, 0] != 0.0
    # rows 1 and 2 still feel steps 0 and 1; nothing from row 3 onwards reaches them
    w2 = np.zeros((n, 5)); w2[3] = 1.0
    ga2, g02 = _vjp(oracle.DYN_BICYCLE, sim, acts, w2, av=av, clip=(6.0, 0.3))
    assert np.all(ga2[:3] == 0.0) and np.all(g02 == 0.0)


# ---------------------------------------------------------------------------------------
# O15 discretised actions
# ---------------------------------------------------------------------------------------
def test_discretize_hand_cases():
    """Grid of 5 values over [-2, 2] = {-2, -1, 0, 1, 2}: nearest value, ties to the even bin, ends clamp."""
    v = np.array([0.49, 0.51, -0.5, 0.5, 1.5, 7.0, -9.0, 2.0, -2.0, 1.0], np.float32).reshape(1, 1, -1)
    r = oracle.discretize_actions(v, n=[5], lo=[-2.0], hi=[2.0])
    assert r["index"].reshape(-1).tolist() == [2, 3, 2, 2, 4, 4, 0, 4, 0, 3]     # -0.5 -> bin 1.5 -> 2; 0.5 -> 2.5 -> 2; 1.5 -> 3.5 -> 4
    assert r["action"].reshape(-1).tolist() == [0.0, 1.0, 0.0, 0.0, 2.0, 2.0, -2.0, 2.0, -2.0, 1.0]


def test_discretize_joint_index_and_round_trip():
    """Joint index is row-major over the channels; decode(encode(v)) is the nearest grid value, within
    half a step of v inside the range; grid values are fixed points."""
    n, lo, hi = [7, 5, 3], [-3.0, -0.2, -1.0], [3.0, 0.2, 1.0]
    rng = np.random.default_rng(3)
    act = np.stack([rng.uniform(lo[c], hi[c], (4, 6)) for c in range(3)], axis=1).astype(np.float32)     # [4][3][6]
    r = oracle.discretize_actions(act, n, lo, hi)
    step = [(hi[c] - lo[c]) / (n[c] - 1) for c in range(3)]
    per = [np.rint((act[:, c].astype(np.float64) - lo[c]) / step[c]).astype(int) for c in range(3)]
    inside = np.ones(act[:, 0].shape, bool)
    for c in range(3):                                   # away from bin boundaries the float32 decision is the real one
        frac = (act[:, c].astype(np.float64) - lo[c]) / step[c]
        inside &= np.abs(frac - np.floor(frac) - 0.5) > 1e-4
    joint = (per[0] * n[1] + per[1]) * n[2] + per[2]
    assert np.array_equal(r["index"][inside], joint[inside])
    for c in range(3):
        assert np.all(np.abs(r["action"][:, c] - act[:, c]) <= step[c] / 2 + 1e-6)
    back = oracle.actions_from_index(r["index"], 3, n, lo, hi)
    assert np.array_equal(back, r["action"])
    again = oracle.discretize_actions(back, n, lo, hi)
    assert np.array_equal(again["index"], r["index"]) and np.array_equal(again["action"], back)


def test_discretize_invalid_and_single_bin():
    act = np.array([[[0.3, 0.3]], [[5.0, 5.0]]], np.float32).reshape(1, 2, 2)      # [1][C=2][A=2]
    valid = np.array([[1, 0]], np.uint8)
    r = oracle.discretize_actions(act, n=[3, 1], lo=[0.0, 4.0], hi=[1.0, 4.0], valid=valid)
    assert r["index"].tolist() == [[1, -1]]                      # 0.3 -> 0.5 (bin 1); the single-bin channel adds nothing
    assert r["action"][0, :, 0].tolist() == [0.5, 4.0] and r["action"][0, :, 1].tolist() == [0.0, 0.0]
    assert oracle.actions_from_index(r["index"], 2, [3, 1], [0.0, 4.0], [1.0, 4.0])[0, :, 1].tolist() == [0.0, 0.0]



def test_index_outside_the_grid_decodes_to_the_zero_action():
    """D45: 3 x 2 bins; indices -1, 6 (= total), 7 and INT_MAX are no bins and give 0, never a wrapped bin; 0 .. 5 by hand."""
    idx = np.array([[0, 1, 2, 3, 4, 5, -1, 6, 7, 2**31 - 1]], np.int32)
    back = oracle.actions_from_index(idx, 2, [3, 2], [0.0, 10.0], [1.0, 20.0])
    assert back[0, 0].tolist() == [0.0, 0.0, 0.5, 0.5, 1.0, 1.0, 0.0, 0.0, 0.0, 0.0]
    assert back[0, 1].tolist() == [10.0, 20.0, 10.0, 20.0, 10.0, 20.0, 0.0, 0.0, 0.0, 0.0]

# ---------------------------------------------------------------------------------------
# O7 with order = 1: sorted by distance
# ---------------------------------------------------------------------------------------
def test_topk_sorted_by_distance_matches_numpy_and_the_index_order_set():
    rng = np.random.default_rng(11)
    R, k = 400, 37
    pts = rng.uniform(-50, 50, (R, 2))
    rg = mk_roadgraph([pts])
    rg["valid"][0, rng.choice(R, 40, replace=False)] = 0
    sim = mk_traj(1, 1, 2, valid=1)
    set_agent(sim, 0, 0, 0, 3.0, -4.0, 0.8)
    set_agent(sim, 0, 0, 1, -20.0, 10.0, -2.0)
    a = oracle.observe_topk(sim, rg, 0, k, order=0)
    s = oracle.observe_topk(sim, rg, 0, k, order=1)
    for e in range(2):
        ex, ey = np.float32(sim["x"][0, 0, e]), np.float32(sim["y"][0, 0, e])
        dx = rg["x"][0] - ex; dy = rg["y"][0] - ey
        key = (dy.astype(np.float64) ** 2 + dx.astype(np.float64) ** 2)
        order = np.lexsort((np.arange(R), np.where(rg["valid"][0] != 0, key, np.inf)))[:k]
        assert np.array_equal(s["rg_index"][0, e], order)
        assert np.array_equal(np.sort(s["rg_index"][0, e]), a["rg_index"][0, e])
        # the features travel with their point
        pos = {int(i): j for j, i in enumerate(a["rg_index"][0, e])}
        perm = [pos[int(i)] for i in s["rg_index"][0, e]]
        assert np.array_equal(s["rg_feat"][0, e], a["rg_feat"][0, e][:, perm])
        assert np.array_equal(s["rg_type"][0, e], a["rg_type"][0, e][perm])


def test_topk_sorted_ties_go_to_the_lower_index_and_padding_stays_last():
    """Lattice points on one circle around the ego tie exactly: they come out in ascending index."""
    pts = np.array([(3, 4), (-3, 4), (5, 0), (0, -5), (4, 3), (1, 0), (-4, -3), (10, 0)], float)
    rg = mk_roadgraph([pts])
    sim = mk_traj(1, 1, 1, valid=1)
    set_agent(sim, 0, 0, 0, 0.0, 0.0, 0.0)
    s = oracle.observe_topk(sim, rg, 0, 10, order=1)
    assert s["rg_index"][0, 0].tolist() == [5, 0, 1, 2, 3, 4, 6, 7, -1, -1]
