"""-m gpu edge-case parity: roadgraphs unlike the generators' tidy streets (the nested grids, their
crowded-cell and off-grid fallbacks, zero-length segments, empty scenarios), map coordinates far from the
origin (float32 slack of the cell assignment), egos far off the map for the top-k."""
import numpy as np
import pytest
import torch

import oracle
import paper_2310_08710_b200 as wm
from gpu_util import dev, host, gpu_offroad, compare_offroad
from util import mk_traj, set_agent

pytestmark = pytest.mark.gpu


def soup_roadgraph(rng, B, R, offset):
    """Random short polylines that cross each other, isolated points, exact duplicates, lane points and
    invalid points mixed in; scenario 0 has no road edge at all; the last scenario is one dense knot."""
    rg = {"x": np.zeros((B, R), np.float32), "y": np.zeros((B, R), np.float32), "dir_x": np.ones((B, R), np.float32),
          "dir_y": np.zeros((B, R), np.float32), "type": np.ones((B, R), np.int32), "id": np.zeros((B, R), np.int32),
          "valid": np.zeros((B, R), np.uint8)}
    for b in range(B):
        i, pid = 0, 0
        span = 3.0 if b == B - 1 else 150.0                      # the knot: everything within 3 m -> crowded cells
        while i < R - 40:
            n = int(rng.integers(1, 30))
            p0 = rng.uniform(0, span, 2) + offset
            th = rng.uniform(-np.pi, np.pi); step = rng.uniform(0.05, 2.0)
            th_s = th + np.cumsum(rng.normal(0, 0.3, n))
            pts = p0 + np.cumsum(np.stack([np.cos(th_s), np.sin(th_s)], 1) * step, 0)
            if rng.random() < 0.2 and n > 3:
                pts[2] = pts[1]                                  # exact duplicate -> zero-length segment (D29)
            typ = 2 if (b > 0 and rng.random() < 0.7) else 1
            rg["x"][b, i:i + n] = pts[:, 0]; rg["y"][b, i:i + n] = pts[:, 1]
            d = rng.normal(size=(n, 2)); d /= np.linalg.norm(d, axis=1, keepdims=True)
            rg["dir_x"][b, i:i + n] = d[:, 0]; rg["dir_y"][b, i:i + n] = d[:, 1]
            rg["type"][b, i:i + n] = typ; rg["id"][b, i:i + n] = pid; rg["valid"][b, i:i + n] = 1
            if rng.random() < 0.3:
                rg["valid"][b, i + int(rng.integers(0, n))] = 0  # a hole splits the polyline
            i += n; pid += 1
    return rg


@pytest.mark.parametrize("offset", [0.0, 3000.0, -7000.0])
def test_offroad_on_polyline_soup(offset):
    rng = np.random.default_rng(int(abs(offset)) + 1)
    B, A, R = 5, 160, 3000
    rg = soup_roadgraph(rng, B, R, offset)
    tr = mk_traj(B, 1, A)
    for b in range(B):
        for a in range(A):
            far = a % 9 == 0
            c = rng.uniform(-400, 550, 2) if far else rng.uniform(-10, 160, 2)
            if b == B - 1 and not far:
                c = rng.uniform(-4, 7, 2)
            set_agent(tr, b, 0, a, c[0] + offset, c[1] + offset, rng.uniform(-4, 4), 0, 0, rng.uniform(0.5, 12), rng.uniform(0.4, 3), valid=int(a % 11 != 0))
    stats = []
    for mode in (wm.WM_OFFROAD_CULLED, wm.WM_OFFROAD_BRUTE_FORCE):
        h = wm.wm_create(offroad_mode=mode)
        tr_d, rg_d = dev(tr), dev(rg)
        wm.wm_prepare(h, rg_d)
        sd, cd, fl = gpu_offroad(h, tr_d, 0)
        orc = oracle.offroad(tr, 0, rg)
        # scenario 0 has no road-edge segment: -FLT_MAX, flag 0 (D20)
        v0 = tr["valid"][0, 0] == 1
        assert np.all(sd[0][v0] == -np.finfo(np.float32).max) and fl[0].sum() == 0
        # float32 coordinates: one ulp of |offset| + 200 m enters every distance (DESIGN.md tolerances)
        ulp = float(np.spacing(np.float32(abs(offset) + 700.0)))
        sub = lambda d, sl: {k: (v[sl] if v is not None else None) for k, v in d.items()}
        err = np.abs(np.abs(cd[1:].astype(np.float64)) - np.abs(orc["corner_dist"][1:].astype(np.float64)))
        vc = np.broadcast_to((tr["valid"][1:, 0] == 1)[:, None, :], err.shape)
        assert err[vc].max() <= 1e-5 * np.abs(orc["corner_dist"][1:][vc]).max() + 3e-6 + 4 * ulp
        if offset == 0.0:
            stats.append(compare_offroad(sd[1:], cd[1:], fl[1:], sub(orc, slice(1, None)), tr["valid"][1:, 0]))
        if mode == wm.WM_OFFROAD_CULLED:
            first = (sd.copy(), fl.copy(), cd.copy())
        else:
            # Both searches use the same per-pair arithmetic; the grid additionally drops a segment that its
            # neighbour on the polyline beats in exact arithmetic (rules P / N), and at such a shared vertex the
            # two float32 distances can differ by an ulp: same result to 2 ulp, same flags away from zero.
            for g0, g1 in ((first[0], sd), (first[2], cd)):
                with np.errstate(over="ignore"):                 # spacing(FLT_MAX) of the empty scenario
                    assert np.all(np.abs(g0 - g1) <= 2 * np.spacing(np.maximum(np.abs(g0), np.abs(g1))))
            assert (np.abs(first[2] - cd) > 0).mean() < 1e-2
            assert np.array_equal(first[1][np.abs(sd) > 1e-4], fl[np.abs(sd) > 1e-4])
        wm.wm_destroy(h)
    if stats:
        print("soup:", stats[0])


def test_topk_egos_far_off_the_map_and_sparse_points():
    rng = np.random.default_rng(9)
    B, A, R, k = 3, 40, 4000, 64
    rg = soup_roadgraph(rng, B, R, 0.0)
    rg["valid"][1, 50:] = 0                                       # scenario 1: only a handful of valid points (< k)
    tr = mk_traj(B, 11, A)
    for b in range(B):
        for a in range(A):
            c = rng.uniform(-3000, 3000, 2) if a % 3 == 0 else rng.uniform(-20, 170, 2)
            for t in range(11):
                set_agent(tr, b, t, a, c[0], c[1], rng.uniform(-3, 3), 1.0, 0.0, valid=int(a % 7 != 0))
    h = wm.wm_create(topk=k)
    tr_d, rg_d = dev(tr), dev(rg)
    wm.wm_prepare(h, rg_d)
    idx = torch.full((B, A, k), 7, dtype=torch.int32, device="cuda"); feat = torch.full((B, A, 4, k), 7.0, device="cuda")
    typ = torch.full((B, A, k), 7, dtype=torch.int32, device="cuda")
    wm.wm_observe(h, tr_d, rg_d, 10, None, None, idx, feat, typ)
    torch.cuda.synchronize()
    o = oracle.observe_topk(tr, rg, 10, k)
    assert np.array_equal(idx.cpu().numpy(), o["rg_index"])
    assert np.array_equal(typ.cpu().numpy(), o["rg_type"])
    assert np.allclose(feat.cpu().numpy(), o["rg_feat"], rtol=1e-5, atol=2e-3)     # ego-frame coordinates up to 6 km in float32
    wm.wm_destroy(h)


@pytest.mark.parametrize("mode", ["culled", "brute"])
def test_exact_tie_between_stored_segments_63_and_64(mode):
    """D17 (ties -> lower index) where the brute-force scan keeps its segments interleaved over the lanes: stored
    segments 63 and 64 of a tile sit in lanes 31 and 0.  A polyline runs east along y = 0 to the vertex (64, 0) and
    turns back by 135 degrees; the box corner (66, 1) is nearest to that vertex on BOTH segments (d2 = 5 exactly, all
    coordinates are small integers), left of segment 63 and right of segment 64: the lower index, 63, must give
    the sign (negative = on-road).  The oracle marks the corner ambiguous, so the generic comparisons skip it."""
    from util import mk_roadgraph
    pts = [(float(i), 0.0) for i in range(65)] + [(59.0, 5.0)]
    rg = mk_roadgraph([np.array(pts)], B=1, R=128)
    tr = mk_traj(1, 1, 32)
    set_agent(tr, 0, 0, 0, 65.0, 0.0, 0.0, 0, 0, 2.0, 2.0)
    orc = oracle.offroad(tr, 0, rg)
    k = 0                                                         # D30: corner 0 = front-left = (66, 1)
    assert orc["win_seg"][0, k, 0] == 63 and orc["ambig"][0, k, 0] == 1
    assert orc["corner_dist"][0, k, 0] == -np.float32(np.sqrt(np.float32(5.0)))
    h = wm.wm_create(offroad_mode=wm.WM_OFFROAD_CULLED if mode == "culled" else wm.WM_OFFROAD_BRUTE_FORCE)
    tr_d, rg_d = dev(tr), dev(rg)
    wm.wm_prepare(h, rg_d)
    sd, cd, fl = gpu_offroad(h, tr_d, 0)
    assert cd[0, k, 0] == orc["corner_dist"][0, k, 0], (cd[0, :, 0], orc["corner_dist"][0, :, 0])
    wm.wm_destroy(h)


def test_oversize_shapes_are_refused_not_launched():
    """wm.h "Limits": A <= 1024 agents, B <= 65 535 scenarios per call.  Every entry point that launches over
    (scenario, agent) returns WM_ERR_UNSUPPORTED for a shape beyond them - not WM_ERR_CUDA from a launch the
    hardware rejected - before touching its outputs."""
    def traj(B, T, A):
        tr = {k: torch.zeros((B, T, A), device="cuda") for k in wm.TRAJ_F}
        tr["valid"] = torch.ones((B, T, A), dtype=torch.uint8, device="cuda")
        return tr
    def paths(B, A, P=2):
        return dict(x=torch.zeros((B, A, P), device="cuda"), y=torch.zeros((B, A, P), device="cuda"),
                    arc_len=torch.zeros((B, A, P), device="cuda"), valid=torch.ones((B, A, P), dtype=torch.uint8, device="cuda"))
    h = wm.wm_create(history=1)
    for B, A in ((1, 1025), (65536, 1)):
        T, n = 3, 1
        tr, sim = traj(B, T, A), traj(B, T, A)
        f = lambda *s: torch.full(s, 7.0, device="cuda")
        u = lambda *s: torch.full(s, 7, dtype=torch.uint8, device="cuda")
        act, av = f(B, n, 2, A), u(B, n, A)
        out = wm.alloc_rollout_out(B, n, A)
        pa = paths(B, A)
        calls = {
            "wm_reset": lambda: wm.wm_reset(h, tr, sim),
            "wm_step": lambda: wm.wm_step(h, tr, sim, 0, act[:, 0].contiguous(), av[:, 0].contiguous()),
            "wm_metrics_overlap": lambda: wm.wm_metrics_overlap(h, sim, 0, None, u(B, A)),
            "wm_log_divergence": lambda: wm.wm_log_divergence(h, tr, sim, 0, f(B, A), u(B, A)),
            "wm_expert_actions": lambda: wm.wm_expert_actions(h, tr, 0, n, f(B, n, 2, A), u(B, n, A)),
            "wm_metrics_kinematic": lambda: wm.wm_metrics_kinematic(h, sim, 1, n, f(B, n, A), f(B, n, A), u(B, n, A)),
            "wm_rollout_vjp": lambda: wm.wm_rollout_vjp(h, sim, 0, n, act, av, f(B, n, 5, A), f(B, n, 2, A)),
            "wm_metrics_route_progress": lambda: wm.wm_metrics_route_progress(h, tr, sim, 0, pa, f(B, A), u(B, A)),
            "wm_metrics_offroute": lambda: wm.wm_metrics_offroute(h, sim, 0, pa, None, 5.0, 1.0, f(B, A), u(B, A)),
            "wm_idm_step": lambda: wm.wm_idm_step(h, sim, 0, pa, u(B, A)),
            "wm_observe": lambda: wm.wm_observe(h, sim, None, 0, f(B, A, 1, 7, A), u(B, A, 1, A)),
            "wm_rollout": lambda: wm.wm_rollout(h, tr, sim, 0, n, act, av, out),
            "wm_rollout_kernel_times": lambda: wm.wm_rollout_kernel_times(h, tr, sim, 0, n, act, av, out),
        }
        for name, call in calls.items():
            with pytest.raises(wm.WmError, match="WM_ERR_UNSUPPORTED"):
                call()
        torch.cuda.synchronize()
        assert float(out["ade"].abs().sum()) == 0.0
    wm.wm_destroy(h)


def test_grid_stats_counts_cells_without_a_list():
    """wm_grid_stats: cell counts follow the grid geometry (4 inner per mid cell); an ordinary street map leaves (almost)
    no cell without a list, the 0.1 m-spaced boundary of config 4 leaves many - and the results stay exact there
    (test_gpu_fullsize checks config 4 against the oracle)."""
    import wm_scenarios as ws
    h = wm.wm_create()
    with pytest.raises(wm.WmError, match="STATE"):
        wm.wm_grid_stats(h)
    shares = {}
    for cid, kw in ((1, {}), (4, {"B": 2})):
        cfg = ws.make_config(cid, **kw)
        wm.wm_prepare(h, dev(cfg["roadgraph"]))
        st = wm.wm_grid_stats(h)
        assert st == wm.wm_grid_stats(h)                           # the counters are cleared on every call
        (ni, ci, _), (nm, cm, _), (no, co, _) = st["inner"], st["mid"], st["outer"]
        assert ni > 0 and ni == 4 * nm and no > 0 and 0 <= ci <= ni and 0 <= cm <= nm and 0 <= co <= no
        assert ci >= 4 * cm                                        # the children of a cell without a list have none either
        shares[cid] = st["inner"][2]
        print("config %d: cells without a candidate list: inner %.4f, mid %.4f, outer %.4f" % (cid, st["inner"][2], st["mid"][2], st["outer"][2]))
    assert shares[1] < 0.01
    wm.wm_destroy(h)
