"""-m gpu parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(wm_rollout graph / single calls on the whole batch).  The oracle cannot run the full batches in
test time, so seeded samples of scenarios / egos are checked element by element and the rest
through properties that hold at any size."""
import numpy as np
import pytest
import torch

import oracle
import wm_scenarios as ws
import paper_2310_08710_b200 as wm
from gpu_util import (dev, host, row_of, assert_state_close, compare_offroad, compare_overlap, gpu_offroad,
                      gpu_overlap, DIST_REL, DIST_ABS)

pytestmark = pytest.mark.gpu


def _sub(d, idx):
    return {k: np.ascontiguousarray(v[idx]) for k, v in d.items()}


def test_config5_full_rollout_sampled():
    """B=4096, A=128, R=20000, T=91, 80-step bicycle rollout in one CUDA graph (bench.py's job)."""
    cfg = ws.make_config(5)
    log, rg = cfg["log"], cfg["roadgraph"]
    B, T, A = log["x"].shape
    assert (B, T, A) == (4096, 91, 128) and rg["x"].shape[1] == 20000
    n = 80
    h = wm.wm_create()
    log_d, rg_d = dev(log), dev(rg)
    assert wm.wm_prepare(h, rg_d) == 6534
    sim_d = wm.empty_traj_like(log_d)
    t0 = wm.wm_reset(h, log_d, sim_d)
    out_d = wm.alloc_rollout_out(B, n, A)
    acts_d, av_d = torch.from_numpy(cfg["actions"]).cuda(), torch.from_numpy(cfg["action_valid"]).cuda()
    wm.wm_rollout(h, log_d, sim_d, t0, n, acts_d, av_d, out_d)
    wm.wm_reset(h, log_d, sim_d)
    wm.wm_rollout(h, log_d, sim_d, t0, n, acts_d, av_d, out_d)          # graph replay, as in the bench
    torch.cuda.synchronize()
    # ---- properties over the whole batch ----
    valid = sim_d["valid"][:, t0 + 1:t0 + 1 + n]
    assert torch.equal(out_d["any_overlap"], out_d["overlap"].amax(dim=1))
    assert torch.equal(out_d["any_offroad"], out_d["offroad"].amax(dim=1))
    assert int(out_d["offroad"][valid == 0].sum()) == 0 and int(out_d["overlap"][valid == 0].sum()) == 0
    assert bool(torch.isfinite(out_d["offroad_dist"]).all()) and bool(torch.isfinite(out_d["log_div"]).all())
    assert torch.equal(out_d["offroad"] == 1, (out_d["offroad_dist"] > 0) & (valid == 1))
    ctrl = (av_d == 1) & (sim_d["valid"][:, t0:t0 + n] == 1)
    assert bool((valid[ctrl] == 1).all())                                # D9
    assert bool(torch.isfinite(sim_d["x"][:, t0 + 1:t0 + 1 + n][valid == 1]).all())
    assert 0.02 < float(out_d["offroad"].float().mean()) < 0.9
    # ---- sampled scenarios against the oracle ----
    rng = np.random.default_rng(20231008)
    idx = np.sort(rng.choice(B, 64, replace=False))
    got = {k: v[idx].cpu().numpy() for k, v in sim_d.items()}
    out = {k: v[idx].cpu().numpy() for k, v in out_d.items()}
    lg, rgs = _sub(log, idx), _sub(rg, idx)
    sim_o = oracle.reset(lg)
    oracle.rollout(lg, sim_o, rgs, t0, n, oracle.DYN_BICYCLE, np.ascontiguousarray(cfg["actions"][idx]),
                   np.ascontiguousarray(cfg["action_valid"][idx]))
    assert_state_close(row_of(got, t0 + 1), row_of(sim_o, t0 + 1))
    assert_state_close(row_of(got, t0 + n), row_of(sim_o, t0 + n), pos_tol=1e-3, yaw_tol=1e-4, vel_tol=1e-2)
    n_amb = 0
    for s in (0, 9, 17, 29, 41, 55, 68, 79):                             # teacher-forced metrics (P16)
        t = t0 + s + 1
        vq = got["valid"][:, t] == 1
        off = oracle.offroad(got, t, rgs)
        clean = vq & ~(off["ambig"] == 1).any(axis=1)
        n_amb += int(((off["ambig"] == 1) & vq[:, None, :]).sum())
        assert np.array_equal(out["offroad"][:, s][clean], off["flag"][clean])
        err = np.abs(out["offroad_dist"][:, s][clean].astype(np.float64) - off["signed_dist"][clean])
        assert (err <= DIST_REL * np.abs(off["signed_dist"][clean]) + DIST_ABS).all()
        ov = oracle.overlap(got, t, want_pair=False)
        cl = ~(np.abs(ov["gap"]) < 1e-4).any(axis=2)
        assert np.array_equal(out["overlap"][:, s][cl], ov["flag"][cl])
        ld = oracle.log_divergence(lg, got, t)
        assert np.allclose(out["log_div"][:, s], ld["dist"], rtol=1e-5, atol=1e-6)
    print("config5 full: sampled scenarios %s, ambiguous corners %d" % (idx.tolist(), n_amb))
    wm.wm_destroy(h)


def test_config2_full_single_step_sampled():
    """B=512, A=128, R=30000: one DeltaLocal step, then overlap, offroad, log divergence."""
    cfg = ws.make_config(2)
    log, rg = cfg["log"], cfg["roadgraph"]
    B, T, A = log["x"].shape
    assert (B, A) == (512, 128) and rg["x"].shape[1] == 30000
    h = wm.wm_create(dynamics=wm.WM_DYN_DELTA_LOCAL)
    log_d, rg_d = dev(log), dev(rg)
    assert wm.wm_prepare(h, rg_d) == 9900
    sim_d = wm.empty_traj_like(log_d)
    t = wm.wm_reset(h, log_d, sim_d)
    act = np.ascontiguousarray(cfg["actions"][:, 0]); av = np.ascontiguousarray(cfg["action_valid"][:, 0])
    wm.wm_step(h, log_d, sim_d, t, torch.from_numpy(act).cuda(), torch.from_numpy(av).cuda())
    sd, cd, fl = gpu_offroad(h, sim_d, t + 1)
    pair, ofl = gpu_overlap(h, sim_d, t + 1)
    rng = np.random.default_rng(2)
    idx = np.sort(rng.choice(B, 8, replace=False))
    got = {k: v[idx].cpu().numpy() for k, v in sim_d.items()}
    lg, rgs = _sub(log, idx), _sub(rg, idx)
    sim_o = oracle.reset(lg)
    oracle.step(lg, sim_o, t, oracle.DYN_DELTA_LOCAL, act[idx], av[idx])
    assert_state_close(row_of(got, t + 1), row_of(sim_o, t + 1))
    st = compare_offroad(sd[idx], cd[idx], fl[idx], oracle.offroad(got, t + 1, rgs), got["valid"][:, t + 1])
    so = compare_overlap(pair[idx], ofl[idx], oracle.overlap(got, t + 1), got["valid"][:, t + 1])
    print("config2 full:", st, so)
    v = sim_d["valid"][:, t + 1].cpu().numpy() == 1
    assert np.all(sd[~v] == 0) and np.all(fl[~v] == 0) and np.isfinite(sd).all()
    wm.wm_destroy(h)


def test_config4_full_overlap_and_offroad():
    """B=64, A=512 crowded lot: pairwise SAT and offroad on the whole batch against the oracle."""
    cfg = ws.make_config(4)
    log, rg = cfg["log"], cfg["roadgraph"]
    assert log["x"].shape == (64, 1, 512) and rg["x"].shape == (64, 5000)
    for mode in (wm.WM_OFFROAD_CULLED, wm.WM_OFFROAD_BRUTE_FORCE):
        h = wm.wm_create(offroad_mode=mode)
        log_d, rg_d = dev(log), dev(rg)
        assert wm.wm_prepare(h, rg_d) == 4999
        sd, cd, fl = gpu_offroad(h, log_d, 0)
        st = compare_offroad(sd, cd, fl, oracle.offroad(log, 0, rg), log["valid"][:, 0])
        if mode == wm.WM_OFFROAD_CULLED:
            pair, ofl = gpu_overlap(h, log_d, 0)
            so = compare_overlap(pair, ofl, oracle.overlap(log, 0), log["valid"][:, 0])
            print("config4 full:", st, so, "flagged offroad %d" % int(fl.sum()))
            assert so["overlap_frac"] > 0.002
        wm.wm_destroy(h)


def test_config3_full_observation_sampled():
    """B=256, A=128, R=30000, every valid agent an ego, H=11, k=1000."""
    cfg = ws.make_config(3)
    log, rg = cfg["log"], cfg["roadgraph"]
    B, T, A = log["x"].shape
    assert (B, A) == (256, 128) and rg["x"].shape[1] == 30000
    k, H, t = 1000, 11, 10
    h = wm.wm_create(topk=k)
    log_d, rg_d = dev(log), dev(rg)
    wm.wm_prepare(h, rg_d)
    hist = torch.empty((B, A, H, 7, A), device="cuda"); hv = torch.empty((B, A, H, A), dtype=torch.uint8, device="cuda")
    idx = torch.empty((B, A, k), dtype=torch.int32, device="cuda")
    feat = torch.empty((B, A, 4, k), device="cuda"); typ = torch.empty((B, A, k), dtype=torch.int32, device="cuda")
    wm.wm_observe(h, log_d, rg_d, t, hist, hv, idx, feat, typ)
    torch.cuda.synchronize()
    # properties on everything
    valid_e = torch.from_numpy(log["valid"][:, t]).cuda() == 1
    assert bool((idx[valid_e] >= 0).all()) and bool((idx[~valid_e] == -1).all())
    assert bool((idx[valid_e][:, 1:] > idx[valid_e][:, :-1]).all())              # ascending, distinct
    assert bool((hv[~valid_e] == 0).all()) and bool((hist[~valid_e] == 0).all())
    assert bool(torch.isfinite(hist).all()) and bool(torch.isfinite(feat).all())
    # sampled scenarios against the oracle
    rng = np.random.default_rng(3)
    sel = np.sort(rng.choice(B, 3, replace=False))
    lg, rgs = _sub(log, sel), _sub(rg, sel)
    ok = oracle.observe_topk(lg, rgs, t, k)
    assert np.array_equal(idx[sel].cpu().numpy(), ok["rg_index"])
    assert np.array_equal(typ[sel].cpu().numpy(), ok["rg_type"])
    assert np.allclose(feat[sel].cpu().numpy(), ok["rg_feat"], rtol=1e-5, atol=2e-4)
    oh = oracle.observe_history(lg, t, H)
    assert np.array_equal(hv[sel].cpu().numpy(), oh["hist_valid"])
    hg = hist[sel].cpu().numpy()
    for f in (0, 1, 3, 4, 5, 6):
        assert np.allclose(hg[:, :, :, f], oh["hist"][:, :, :, f], rtol=1e-5, atol=1e-4), f
    d = np.abs(np.angle(np.exp(1j * (hg[:, :, :, 2].astype(np.float64) - oh["hist"][:, :, :, 2]))))
    assert d.max() < 1e-5                                                        # yaw modulo 2 pi
    wm.wm_destroy(h)
