"""The seeded generators: shapes, determinism per scenario, and the recipe's stated structure."""
import numpy as np

import wm_scenarios as ws


def test_config1_shapes_and_recipe():
    c = ws.make_config(1)
    assert c["log"]["x"].shape == (4, 91, 32) and c["roadgraph"]["x"].shape == (4, 2000)
    assert c["actions"].shape == (4, 80, 2, 32) and c["action_valid"].shape == (4, 80, 32)
    rg = c["roadgraph"]
    assert (rg["type"] == ws.TYPE_ROAD_EDGE).sum() == 4 * 20 * 66 and (rg["type"] == ws.TYPE_LANE).sum() == 4 * 20 * 34
    a = c["actions"]
    assert a[:, :, 0].min() >= -3 and a[:, :, 0].max() <= 3 and np.abs(a[:, :, 1]).max() <= 0.1
    v = c["log"]["valid"][:, 10] == 1
    assert np.isnan(c["log"]["x"][:, 10][~v]).all() and not np.isnan(c["log"]["x"][:, 10][v]).any()
    sp = np.hypot(c["log"]["vel_x"][:, 0][v], c["log"]["vel_y"][:, 0][v])
    assert sp.max() <= 15.0 and 4.0 <= c["log"]["length"][:, 0][v].min() and c["log"]["width"][:, 0][v].max() <= 2.2
    # unit directions, 0.5 m spacing on centrelines
    assert np.allclose(np.hypot(rg["dir_x"], rg["dir_y"]), 1.0, atol=1e-6)


def test_street_configs_are_per_scenario_deterministic():
    a = ws.make_config(5, B=6, n_steps=3)
    b = ws.make_config(5, b_ids=[4, 1], n_steps=3)
    for k in a["log"]:
        assert np.array_equal(a["log"][k][4], b["log"][k][0], equal_nan=True)
        assert np.array_equal(a["log"][k][1], b["log"][k][1], equal_nan=True)
    for k in a["roadgraph"]:
        assert np.array_equal(a["roadgraph"][k][4], b["roadgraph"][k][0])
    assert np.array_equal(a["actions"][4], b["actions"][0])
    assert not np.array_equal(a["roadgraph"]["x"][0], a["roadgraph"]["x"][1])     # distinct roadgraphs


def test_street_roadgraph_structure():
    c = ws.make_config(2, B=3)
    rg = c["roadgraph"]
    assert rg["x"].shape == (3, 30000) and rg["valid"].sum() == 3 * 30000
    edge = rg["type"] == ws.TYPE_ROAD_EDGE
    assert edge.sum() == 3 * 10000                                       # exactly 1/3 road edge
    c5 = ws.make_config(5, B=2, n_steps=1)
    rg5 = c5["roadgraph"]
    assert rg5["valid"][0].sum() == 19800 and rg5["valid"][0, 19800:].sum() == 0   # 200 trailing invalid
    # spacing 0.5 m within a polyline
    same = rg["id"][0, 1:] == rg["id"][0, :-1]
    d = np.hypot(np.diff(rg["x"][0].astype(np.float64)), np.diff(rg["y"][0].astype(np.float64)))
    assert np.allclose(d[same], 0.5, atol=1e-4)
    # agent mix and validity
    v = c["log"]["valid"][:, 0]
    L = c["log"]["length"][:, 0]
    veh = (L >= 4.0) & (v == 1); ped = (L <= 1.0) & (v == 1)
    assert 0.55 < veh.sum() / v.sum() < 0.85 and 0.1 < ped.sum() / v.sum() < 0.3
    assert 0.70 < c["log"]["valid"][:, 10].mean() < 0.9
    assert c["actions"].shape == (3, 1, 3, 128) and np.abs(c["actions"][:, 0, :2]).max() <= 0.5


def test_config4_lot():
    c = ws.make_config(4, B=2)
    assert c["log"]["x"].shape == (2, 1, 512) and c["roadgraph"]["x"].shape == (2, 5000)
    assert (c["roadgraph"]["type"] == ws.TYPE_ROAD_EDGE).all() and (c["log"]["valid"] == 1).all()
    assert c["log"]["x"].min() > -1 and c["log"]["x"].max() < 49 and c["log"]["y"].max() < 193


def test_make_paths_structure():
    """Synthetic on-route paths: logged positions in time order, then a straight extension; arc length
    non-decreasing from 0; agents never logged have no path; deterministic."""
    cfg = ws.make_config(1, n_steps=2)
    log = cfg["log"]
    B, T, A = log["x"].shape
    pa = ws.make_paths(log, extend=16)
    pb = ws.make_paths(log, extend=16)
    for k in pa:
        assert np.array_equal(pa[k], pb[k]) and pa[k].shape == (B, A, T + 16)
    n_logged = (log["valid"] == 1).sum(axis=1)                      # [B][A]
    n_path = (pa["valid"] == 1).sum(axis=2)
    assert np.array_equal(n_path, np.where(n_logged > 0, n_logged + 16, 0))
    v = pa["valid"] == 1
    assert np.all(v[:, :, :-1] >= v[:, :, 1:])                      # valid points form a prefix
    d = np.diff(pa["arc_len"].astype(np.float64), axis=2)
    assert np.all(d[v[:, :, 1:]] >= 0) and np.all(pa["arc_len"][:, :, 0] == 0)
    assert np.isfinite(pa["x"]).all() and np.isfinite(pa["y"]).all()
    # the first point is the first valid logged position
    b, a = np.argwhere(n_logged > 0)[0]
    t0 = int(np.argmax(log["valid"][b, :, a] == 1))
    assert pa["x"][b, a, 0] == log["x"][b, t0, a] and pa["y"][b, a, 0] == log["y"][b, t0, a]
