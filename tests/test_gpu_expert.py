"""-m gpu parity tests of the expert actor (wm_expert_actions; L204, L335, Eq. 3) and the
kinematic-infeasibility metric (wm_metrics_kinematic; L104) against the oracle.

Tolerances: acceleration abs 1e-3 m/s^2 (float32 speeds, ulp(15 m/s)/dt = 1e-5, two square
roots); curvature |d kappa| <= 1e-5 |kappa| + 4e-6 / den + 1e-6 (a float32 heading difference of up to
~2 ulp(yaw) divided by the distance travelled den); delta actions abs 2e-5; flags bit-exact outside the
band where |a| or |kappa| is within its tolerance of the limit (counted)."""
import numpy as np
import pytest
import torch

import oracle
import paper_2310_08710_b200 as wm
import wm_scenarios as ws
from gpu_util import dev, host

from defs_f64 import route_ratio_in_double

pytestmark = pytest.mark.gpu

A_TOL = 1e-3


def k_tol(kappa, den):
    return 1e-5 * np.abs(kappa) + 4e-6 / np.maximum(den, 1e-12) + 1e-6


def _gpu_expert(h, tr_d, t, n, C):
    B, T, A = tr_d["x"].shape
    act = torch.full((B, n, C, A), 7.0, device="cuda"); av = torch.full((B, n, A), 9, dtype=torch.uint8, device="cuda")
    wm.wm_expert_actions(h, tr_d, t, n, act, av)
    torch.cuda.synchronize()
    return act, av


@pytest.mark.parametrize("cid,B", [(1, None), (5, 6)])
def test_expert_actions_match_oracle(cid, B):
    cfg = ws.make_config(cid, n_steps=80) if B is None else ws.make_config(cid, B=B, n_steps=80)
    log = cfg["log"]
    log_d = dev(log)
    for dyn, odyn, C in ((wm.WM_DYN_INVERTIBLE_BICYCLE, oracle.DYN_BICYCLE, 2), (wm.WM_DYN_DELTA_LOCAL, oracle.DYN_DELTA_LOCAL, 3),
                         (wm.WM_DYN_DELTA_GLOBAL, oracle.DYN_DELTA_GLOBAL, 3)):
        h = wm.wm_create(dynamics=dyn)
        act, av = _gpu_expert(h, log_d, 10, 80, C)
        e = oracle.expert_actions(log, 10, 80, odyn)
        assert np.array_equal(av.cpu().numpy(), e["valid"])
        g = act.cpu().numpy().astype(np.float64); r = e["action"].astype(np.float64)
        v = e["valid"] == 1
        assert np.all(g[~np.broadcast_to(v[:, :, None, :], g.shape)] == 0)          # D10
        if C == 2:
            assert np.abs(g[:, :, 0] - r[:, :, 0])[v].max() <= A_TOL
            dk = np.abs(g[:, :, 1] - r[:, :, 1])
            assert np.all(dk[v] <= k_tol(r[:, :, 1], e["kden"])[v]), float((dk - k_tol(r[:, :, 1], e["kden"]))[v].max())
            assert v.sum() > 1000 and np.abs(r[:, :, 1][v]).max() > 0.01
        else:
            assert np.abs(g - r)[np.broadcast_to(v[:, :, None, :], g.shape)].max() <= 2e-5
        wm.wm_destroy(h)


def test_kinematic_metric_matches_oracle_on_a_rollout():
    """Rows of a GPU rollout with actions beyond the limits for some agents (clipping off), so that
    both branches of the flag occur."""
    n = 40
    cfg = ws.make_config(5, B=8, n_steps=n)
    log, rg = cfg["log"], cfg["roadgraph"]
    B, T, A = log["x"].shape
    acts = cfg["actions"].copy()
    acts[:, :, 0, ::5] *= 2.6            # |a| up to 7.8
    acts[:, :, 1, 1::7] *= 4.0           # |kappa| up to 0.4
    h = wm.wm_create(max_accel=0.0, max_curvature=0.0)          # no clipping in the step (D7)
    log_d, rg_d = dev(log), dev(rg)
    sim_d = wm.empty_traj_like(log_d)
    wm.wm_prepare(h, rg_d)
    t0 = wm.wm_reset(h, log_d, sim_d)
    out = wm.alloc_rollout_out(B, n, A)
    wm.wm_rollout(h, log_d, sim_d, t0, n, torch.from_numpy(acts).cuda(), torch.from_numpy(cfg["action_valid"]).cuda(), out)
    hk = wm.wm_create()                                          # the metric's limits: 6, 0.3
    acc = torch.full((B, n, A), 7.0, device="cuda"); cur = torch.full((B, n, A), 7.0, device="cuda")
    fl = torch.full((B, n, A), 9, dtype=torch.uint8, device="cuda")
    wm.wm_metrics_kinematic(hk, sim_d, t0 + 1, n, acc, cur, fl)
    torch.cuda.synchronize()
    sim = host(sim_d)
    k = oracle.kinematic(sim, t0 + 1, n)
    v = k["valid"] == 1
    ga, gk, gf = acc.cpu().numpy().astype(np.float64), cur.cpu().numpy().astype(np.float64), fl.cpu().numpy()
    assert np.all(ga[~v] == 0) and np.all(gk[~v] == 0) and np.all(gf[~v] == 0)
    ra, rk = k["accel"].astype(np.float64), k["curvature"].astype(np.float64)
    kt = k_tol(rk, k["kden"])
    assert np.abs(ga - ra)[v].max() <= A_TOL
    assert np.all(np.abs(gk - rk)[v] <= kt[v])
    band = (np.abs(np.abs(ra) - 6.0) <= A_TOL) | (np.abs(np.abs(rk) - 0.3) <= kt)
    clean = v & ~band
    assert np.array_equal(gf[clean], k["flag"][clean])
    n_flag = int(k["flag"][clean].sum())
    print("kinematic: %d transitions, %d in the band, %d flagged" % (int(v.sum()), int((v & band).sum()), n_flag))
    assert n_flag > 100 and n_flag < clean.sum() // 2
    wm.wm_destroy(h); wm.wm_destroy(hk)


def test_expert_rollouts():
    """RolloutExpert (L200): expert actions of the log, then the rollout.  DeltaLocal reproduces the
    log (Table 3: Log ADE 0.00); the bicycle expert follows the oracle's expert rollout and, by
    construction (L198), stays kinematically feasible wherever the log is."""
    n = 80
    cfg = ws.make_config(5, B=8, n_steps=n)
    log, rg = cfg["log"], cfg["roadgraph"]
    B, T, A = log["x"].shape
    log_d, rg_d = dev(log), dev(rg)
    for dyn, odyn, C in ((wm.WM_DYN_DELTA_LOCAL, oracle.DYN_DELTA_LOCAL, 3), (wm.WM_DYN_DELTA_GLOBAL, oracle.DYN_DELTA_GLOBAL, 3),
                         (wm.WM_DYN_INVERTIBLE_BICYCLE, oracle.DYN_BICYCLE, 2)):
        h = wm.wm_create(dynamics=dyn)
        wm.wm_prepare(h, rg_d)
        sim_d = wm.empty_traj_like(log_d)
        t0 = wm.wm_reset(h, log_d, sim_d)
        act, av = _gpu_expert(h, log_d, t0, n, C)
        out = wm.alloc_rollout_out(B, n, A)
        wm.wm_rollout(h, log_d, sim_d, t0, n, act, av, out)
        torch.cuda.synchronize()
        ade = out["ade"].cpu().numpy()
        e = oracle.expert_actions(log, t0, n, odyn)
        sim_o = oracle.reset(log)
        oo = oracle.rollout(log, sim_o, rg, t0, n, odyn, e["action"], e["valid"])
        sim = host(sim_d)
        assert np.array_equal(sim["valid"], sim_o["valid"])
        v = sim_o["valid"][:, t0 + n] == 1
        if dyn != wm.WM_DYN_INVERTIBLE_BICYCLE:
            assert round(float(ade.max()), 2) == 0.0 and ade.max() < 5e-3
        err = np.hypot(sim["x"][:, t0 + n][v].astype(np.float64) - sim_o["x"][:, t0 + n][v], sim["y"][:, t0 + n][v].astype(np.float64) - sim_o["y"][:, t0 + n][v])
        assert err.max() < 2e-3, float(err.max())
        assert np.abs(ade - oo["ade"]).max() < 2e-3
        wm.wm_destroy(h)


def test_argument_checks():
    cfg = ws.make_config(1, n_steps=4)
    log_d = dev(cfg["log"])
    B, T, A = log_d["x"].shape
    h = wm.wm_create()
    act = torch.zeros((B, 1, 2, A), device="cuda"); av = torch.zeros((B, 1, A), dtype=torch.uint8, device="cuda")
    fl = torch.zeros((B, 1, A), dtype=torch.uint8, device="cuda")
    for bad in (lambda: wm.wm_expert_actions(h, log_d, T - 1, 1, act, av), lambda: wm.wm_expert_actions(h, log_d, -1, 1, act, av),
                lambda: wm.wm_metrics_kinematic(h, log_d, 0, 1, None, None, fl), lambda: wm.wm_metrics_kinematic(h, log_d, T, 1, None, None, fl)):
        with pytest.raises(RuntimeError):
            bad()
    wm.wm_metrics_kinematic(h, log_d, T - 1, 1, None, None, fl)          # NULL accel / curvature are allowed
    torch.cuda.synchronize()
    wm.wm_destroy(h)


def test_route_progress_matches_oracle():
    """wm_metrics_route_progress (L96) on the rows of a GPU rollout, synthetic per-agent paths; the
    closest-point decision is taken in float32 on both sides (D33), so validity and the ratio's
    numerator / denominator indices agree exactly and the ratio to float32 rounding."""
    n = 80
    for cid, B in ((5, 6), (1, None)):
        cfg = ws.make_config(cid, n_steps=n) if B is None else ws.make_config(cid, B=B, n_steps=n)
        log, rg = cfg["log"], cfg["roadgraph"]
        Bn, T, A = log["x"].shape
        paths = ws.make_paths(log)
        paths["valid"][:, ::7, 5] = 0                          # holes in some paths
        h = wm.wm_create()
        log_d, rg_d = dev(log), dev(rg)
        sim_d = wm.empty_traj_like(log_d)
        wm.wm_prepare(h, rg_d)
        t0 = wm.wm_reset(h, log_d, sim_d)
        out = wm.alloc_rollout_out(Bn, n, A)
        wm.wm_rollout(h, log_d, sim_d, t0, n, torch.from_numpy(cfg["actions"]).cuda(), torch.from_numpy(cfg["action_valid"]).cuda(), out)
        paths_d = {k: torch.from_numpy(v).cuda() for k, v in paths.items()}
        sim = None
        for t in (t0, t0 + 37, t0 + n):
            ratio = torch.full((Bn, A), 7.0, device="cuda"); val = torch.full((Bn, A), 9, dtype=torch.uint8, device="cuda")
            wm.wm_metrics_route_progress(h, log_d, sim_d, t, paths_d, ratio, val)
            torch.cuda.synchronize()
            sim = host(sim_d) if sim is None else sim
            r = oracle.route_progress(log, sim, t, paths)
            assert np.array_equal(val.cpu().numpy(), r["valid"])
            g = ratio.cpu().numpy().astype(np.float64)
            assert np.all(g[r["valid"] == 0] == 0)
            v = r["valid"] == 1
            assert np.all(np.abs(g - r["ratio"])[v] <= 1e-5 * np.maximum(1.0, np.abs(r["ratio"][v])))
            assert v.sum() > 0.5 * (sim["valid"][:, t] == 1).sum()
            # the double-precision definition (D33 takes the decision in float32 on both sides above): wherever the
            # closest points are decided by more than 1e-4 m the GPU's ratio is the definition's; the rest is counted
            rd, decided = route_ratio_in_double(log, sim, t, paths)
            chk = decided & v
            assert np.all(np.abs(g - rd)[chk] <= 1e-5 * np.maximum(1.0, np.abs(rd[chk])))
            print("route progress cfg%d t=%d: %d valid agents, %d decided by > 1e-4 m and equal to the float64 definition, %d in the band"
                  % (cid, t, int(v.sum()), int(chk.sum()), int((v & ~decided).sum())))
            assert chk.sum() > 0.5 * v.sum()
        # the reset state sits on its own logged position: progress of agents logged from step 0 at t0 = progress of the log
        wm.wm_destroy(h)


def test_offroute_matches_oracle_bit_for_bit():
    """wm_metrics_offroute (L98, thresholds as arguments): both sides take the closest-point decision, the
    square root and the two comparisons in float32, so distances and flags agree exactly."""
    n = 80
    cfg = ws.make_config(5, B=6, n_steps=n)
    log, rg = cfg["log"], cfg["roadgraph"]
    B, T, A = log["x"].shape
    on = ws.make_paths(log)
    off = {k: np.ascontiguousarray(np.roll(v, 1, axis=1)) for k, v in on.items()}     # another agent's path as the off-route one
    on["valid"][:, ::9, :] = 0                                    # agents without an on-route path
    h = wm.wm_create()
    log_d, rg_d = dev(log), dev(rg)
    sim_d = wm.empty_traj_like(log_d)
    wm.wm_prepare(h, rg_d)
    t0 = wm.wm_reset(h, log_d, sim_d)
    out = wm.alloc_rollout_out(B, n, A)
    wm.wm_rollout(h, log_d, sim_d, t0, n, torch.from_numpy(cfg["actions"]).cuda(), torch.from_numpy(cfg["action_valid"]).cuda(), out)
    on_d = {k: torch.from_numpy(v).cuda() for k, v in on.items()}
    off_d = {k: torch.from_numpy(v).cuda() for k, v in off.items()}
    sim = host(sim_d)
    total = 0
    for t, offp, offd in ((t0 + n, off, off_d), (t0 + 40, None, None)):
        d = torch.full((B, A), 7.0, device="cuda"); f = torch.full((B, A), 9, dtype=torch.uint8, device="cuda")
        wm.wm_metrics_offroute(h, sim_d, t, on_d, offd, 5.0, 1.0, d, f)
        torch.cuda.synchronize()
        r = oracle.offroute(sim, t, on, offp, 5.0, 1.0)
        assert np.array_equal(d.cpu().numpy(), r["dist_on"]) and np.array_equal(f.cpu().numpy(), r["flag"])
        total += int(r["flag"].sum())
        assert 0 < r["flag"].sum() < (sim["valid"][:, t] == 1).sum()
    wm.wm_destroy(h)
