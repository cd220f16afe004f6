"""Pins for the oracle's observation (O6 history transform, O7 top-k) and rollout (O8)."""
import math

import numpy as np
import pytest

import oracle
from util import mk_traj, set_agent, mk_roadgraph, rigid


def _cfg1():
    import wm_scenarios as ws
    return ws.make_config(1, poison_invalid=False)


# P12 (D22)
def test_history_ego_maps_to_origin_and_preserves_geometry():
    cfg = _cfg1()
    tr = cfg["log"]; t = 10; H = 11
    out = oracle.observe_history(tr, t, H)
    hist, hv = out["hist"], out["hist_valid"]
    B, T, A = tr["x"].shape
    valid_t = tr["valid"][:, t] == 1
    for b in range(B):
        for e in np.nonzero(valid_t[b])[0]:
            me = hist[b, e, H - 1, :, e]
            assert abs(me[0]) < 1e-6 and abs(me[1]) < 1e-6 and abs(me[2]) < 1e-6      # pose -> origin
            sp = math.hypot(float(tr["vel_x"][b, t, e]), float(tr["vel_y"][b, t, e]))
            assert me[3] == pytest.approx(sp, abs=1e-5) and abs(me[4]) < 1e-4          # v along +x (v || yaw here)
            assert me[5] == tr["length"][b, t, e] and me[6] == tr["width"][b, t, e]
    # pairwise distances and relative yaws preserved (for one ego, all valid agents, all steps)
    b, e = 0, int(np.nonzero(valid_t[0])[0][0])
    for h in range(H):
        v = hv[b, e, h] == 1
        px = tr["x"][b, t - H + 1 + h][v].astype(np.float64); py = tr["y"][b, t - H + 1 + h][v].astype(np.float64)
        qx = hist[b, e, h, 0][v].astype(np.float64); qy = hist[b, e, h, 1][v].astype(np.float64)
        d0 = np.hypot(px[:, None] - px[None], py[:, None] - py[None])
        d1 = np.hypot(qx[:, None] - qx[None], qy[:, None] - qy[None])
        assert np.allclose(d0, d1, atol=2e-5)
        dy0 = tr["yaw"][b, t - H + 1 + h][v].astype(np.float64)
        dy1 = hist[b, e, h, 2][v].astype(np.float64)
        rel0 = np.angle(np.exp(1j * (dy0[:, None] - dy0[None]))); rel1 = np.angle(np.exp(1j * (dy1[:, None] - dy1[None])))
        assert np.allclose(np.angle(np.exp(1j * (rel0 - rel1))), 0, atol=2e-6)
        assert np.all((dy1 >= -math.pi) & (dy1 < math.pi))
    # applying R(yaw_e), +p_e restores the input to 1e-5
    ex, ey, eth = (float(tr[k][b, t, e]) for k in ("x", "y", "yaw"))
    c, s = math.cos(eth), math.sin(eth)
    h = 3
    v = hv[b, e, h] == 1
    rx = c * hist[b, e, h, 0] - s * hist[b, e, h, 1] + ex
    ry = s * hist[b, e, h, 0] + c * hist[b, e, h, 1] + ey
    assert np.allclose(rx[v], tr["x"][b, t - H + 1 + h][v], atol=2e-5)
    assert np.allclose(ry[v], tr["y"][b, t - H + 1 + h][v], atol=2e-5)
    rvx = c * hist[b, e, h, 3] - s * hist[b, e, h, 4]
    assert np.allclose(rvx[v], tr["vel_x"][b, t - H + 1 + h][v], atol=2e-5)   # velocities rotated only


def test_history_validity_rules():
    cfg = _cfg1()
    tr = cfg["log"]; t = 10; H = 11
    tr["valid"][0, 4, 7] = 0
    out = oracle.observe_history(tr, t, H)
    hv = out["hist_valid"]
    ego_invalid = tr["valid"][:, t] == 0
    assert hv[ego_invalid].sum() == 0 and np.all(out["hist"][ego_invalid] == 0)   # invalid ego -> zeros
    e = int(np.nonzero(tr["valid"][0, t])[0][0])
    assert hv[0, e, 4, 7] == 0 and np.all(out["hist"][0, e, 4, :, 7] == 0)
    exp = (tr["valid"][:, None, t - H + 1:t + 1, :] & tr["valid"][:, t, :, None, None])
    assert np.array_equal(hv, exp)


# ---- P13 top-k (D23-D25) ----
def _ego_at(x, y, yaw=0.0):
    tr = mk_traj(1, 1, 1, valid=1)
    set_agent(tr, 0, 0, 0, x, y, yaw)
    return tr


def test_topk_matches_full_sort_and_k1_is_argmin():
    rng = np.random.default_rng(3)
    pts = rng.uniform(-50, 50, (300, 2))
    rg = mk_roadgraph([pts])
    rg["valid"][0, ::7] = 0
    tr = _ego_at(3.0, -4.0, 0.5)
    px, py = rg["x"][0].astype(np.float64), rg["y"][0].astype(np.float64)
    d = np.hypot(px - 3.0, py + 4.0)
    d[rg["valid"][0] == 0] = np.inf
    order = np.argsort(d, kind="stable")
    for k in (1, 10, 64):
        out = oracle.observe_topk(tr, rg, 0, k)
        assert sorted(out["rg_index"][0, 0].tolist()) == sorted(order[:k].tolist())
        assert np.all(np.diff(out["rg_index"][0, 0]) > 0)        # ascending index (D24)
    assert oracle.observe_topk(tr, rg, 0, 1)["rg_index"][0, 0, 0] == order[0]


def test_topk_exact_ties_go_to_lower_index_and_padding():
    # 12 lattice points on the circle of radius 5 around the ego + farther points; exact ties
    ring = [(3, 4), (4, 3), (-3, 4), (4, -3), (5, 0), (0, 5), (-5, 0), (0, -5), (-4, 3), (3, -4), (-3, -4), (-4, -3)]
    far = [(7, 0), (0, 8), (9, 9)]
    near = [(1, 0)]
    pts = np.array(far[:1] + ring[:6] + near + ring[6:] + far[1:], np.float64) + [10.0, 20.0]
    rg = mk_roadgraph([pts])
    tr = _ego_at(10.0, 20.0)
    out = oracle.observe_topk(tr, rg, 0, 6)
    # nearest is `near` (index 7); then the 5 lowest-index ring points: indices 1..5
    assert out["rg_index"][0, 0].tolist() == [1, 2, 3, 4, 5, 7]
    # k >= #valid: all valid ascending, then -1 padding with zero features (D25)
    rg["valid"][0, 3] = 0
    out = oracle.observe_topk(tr, rg, 0, 20)
    idx = out["rg_index"][0, 0].tolist()
    assert idx[:15] == [i for i in range(16) if i != 3] and idx[15:] == [-1] * 5
    assert np.all(out["rg_feat"][0, 0, :, 15:] == 0) and np.all(out["rg_type"][0, 0, 15:] == 0)
    assert np.isnan(out["kth_key"][0, 0])


def test_topk_features_in_ego_frame_and_invalid_ego():
    pts = np.array([[12.0, 20.0], [10.0, 23.0]])
    rg = mk_roadgraph([pts])          # dir of both points = unit((−2,3))
    tr = mk_traj(1, 1, 2, valid=1)
    set_agent(tr, 0, 0, 0, 10.0, 20.0, math.pi / 2)      # ego facing +y
    set_agent(tr, 0, 0, 1, 0.0, 0.0, 0.0, valid=0)
    out = oracle.observe_topk(tr, rg, 0, 2)
    f = out["rg_feat"][0, 0]
    # world (+2, 0) seen from an ego facing +y is (0, -2); world (0, +3) is (+3, 0)
    assert np.allclose(f[0], [0.0, 3.0], atol=1e-6) and np.allclose(f[1], [-2.0, 0.0], atol=1e-6)
    u = np.array([-2.0, 3.0]) / math.hypot(2, 3)
    assert np.allclose(f[2], [u[1], u[1]], atol=1e-6) and np.allclose(f[3], [-u[0], -u[0]], atol=1e-6)
    assert out["rg_type"][0, 0].tolist() == [2, 2]
    assert out["rg_index"][0, 1].tolist() == [-1, -1] and np.all(out["rg_feat"][0, 1] == 0)


def test_topk_set_invariant_under_rigid_transform():
    cfg = _cfg1()
    tr, rg = cfg["log"], cfg["roadgraph"]
    k = 200
    out = oracle.observe_topk(tr, rg, 10, k)
    tr2, rg2 = rigid(tr, rg, 0.77, -20.0, 35.0)
    out2 = oracle.observe_topk(tr2, rg2, 10, k)
    B, T, A = tr["x"].shape
    n_diff = 0
    for b in range(B):
        px, py = rg["x"][b].astype(np.float64), rg["y"][b].astype(np.float64)
        for e in range(A):
            if not tr["valid"][b, 10, e]:
                continue
            s1, s2 = set(out["rg_index"][b, e].tolist()), set(out2["rg_index"][b, e].tolist())
            if s1 != s2:      # differences may only involve points within the band of the k-th distance
                d = np.hypot(px - float(tr["x"][b, 10, e]), py - float(tr["y"][b, 10, e]))
                dk = math.sqrt(float(out["kth_key"][b, e]))
                for i in s1 ^ s2:
                    assert abs(d[i] - dk) < 1e-4
                n_diff += 1
    assert n_diff < 20


# ---- O8 rollout = 80 x (step, metrics); ADE (D21) ----
def test_rollout_equals_stepwise_composition():
    cfg = _cfg1()
    log, rg = cfg["log"], cfg["roadgraph"]
    n = 12
    acts = np.ascontiguousarray(cfg["actions"][:, :n]); av = np.ascontiguousarray(cfg["action_valid"][:, :n])
    sim = oracle.reset(log)
    out = oracle.rollout(log, sim, rg, 10, n, oracle.DYN_BICYCLE, acts, av)
    sim2 = oracle.reset(log)
    B, T, A = log["x"].shape
    dsum = np.zeros((B, A)); cnt = np.zeros((B, A))
    for s in range(n):
        oracle.step(log, sim2, 10 + s, oracle.DYN_BICYCLE, np.ascontiguousarray(acts[:, s]), np.ascontiguousarray(av[:, s]))
        ov = oracle.overlap(sim2, 11 + s, want_gap=False, want_pair=False)
        of = oracle.offroad(sim2, 11 + s, rg, details=False)
        ld = oracle.log_divergence(log, sim2, 11 + s)
        assert np.array_equal(out["overlap"][:, s], ov["flag"])
        assert np.array_equal(out["offroad"][:, s], of["flag"])
        assert np.array_equal(out["offroad_dist"][:, s], of["signed_dist"])
        assert np.array_equal(out["log_div"][:, s], ld["dist"])
        dsum += ld["dist"].astype(np.float64) * ld["valid"]; cnt += ld["valid"]
    for k in log:
        assert np.array_equal(sim[k], sim2[k], equal_nan=True)
    assert np.array_equal(out["any_overlap"], out["overlap"].max(axis=1))
    assert np.array_equal(out["any_offroad"], out["offroad"].max(axis=1))
    ade = np.where(cnt > 0, dsum / np.maximum(cnt, 1), 0)
    assert np.allclose(out["ade"], ade, atol=1e-6)
    assert sim["valid"][:, 10 + n + 1:].sum() == 0          # rows beyond the rollout untouched
