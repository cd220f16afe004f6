"""-m gpu parity of the SURVEY 8(f)(4) variants against the oracle: backward pass of the dynamics
(wm_rollout_vjp / wm_step_vjp), discretised action spaces (L204) and the
sorted-by-distance order of the top-k observation (L82, D44).  Everything goes through the C-ABI."""
import numpy as np
import pytest
import torch

import oracle
import wm_scenarios as ws
import paper_2310_08710_b200 as wm
from gpu_util import dev, host

pytestmark = pytest.mark.gpu

DYN = {"bicycle": (wm.WM_DYN_INVERTIBLE_BICYCLE, oracle.DYN_BICYCLE, 2), "delta_local": (wm.WM_DYN_DELTA_LOCAL, oracle.DYN_DELTA_LOCAL, 3),
       "delta_global": (wm.WM_DYN_DELTA_GLOBAL, oracle.DYN_DELTA_GLOBAL, 3)}


def _rollout(cfgid, dyn, n, B=None, seed_actions=5):
    """GPU rollout of n steps; returns (handle, log, sim rows on the host, actions, mask)."""
    wdyn, odyn, C = DYN[dyn]
    cfg = ws.make_config(cfgid, B=B) if B else ws.make_config(cfgid)
    log, rg = cfg["log"], cfg["roadgraph"]
    Bn, T, A = log["x"].shape
    rng = np.random.default_rng(seed_actions)
    if dyn == "bicycle":
        acts = np.stack([rng.uniform(-7, 7, (Bn, n, A)), rng.uniform(-0.35, 0.35, (Bn, n, A))], axis=2).astype(np.float32)   # some beyond the clip limits
    else:
        acts = np.stack([rng.uniform(-0.5, 0.5, (Bn, n, A)), rng.uniform(-0.5, 0.5, (Bn, n, A)), rng.uniform(-0.1, 0.1, (Bn, n, A))], axis=2).astype(np.float32)
    av = (rng.uniform(size=(Bn, n, A)) < 0.9).astype(np.uint8)              # 10 % playback slots
    h = wm.wm_create(dynamics=wdyn)
    log_d, rg_d = dev(log), dev(rg)
    sim_d = wm.empty_traj_like(log_d)
    wm.wm_prepare(h, rg_d)
    t0 = wm.wm_reset(h, log_d, sim_d)
    out_d = wm.alloc_rollout_out(Bn, n, A)
    acts_d, av_d = torch.from_numpy(acts).cuda(), torch.from_numpy(av).cuda()
    wm.wm_rollout(h, log_d, sim_d, t0, n, acts_d, av_d, out_d)
    torch.cuda.synchronize()
    return h, sim_d, host(sim_d), t0, acts, av, acts_d, av_d, odyn, C


@pytest.mark.parametrize("cfgid,dyn,n,B", [(1, "bicycle", 80, None), (5, "bicycle", 40, 24), (2, "delta_local", 12, 16), (2, "delta_global", 12, 16)])
def test_rollout_vjp_matches_oracle(cfgid, dyn, n, B):
    """Teacher-forced on the GPU's own rows: both sides differentiate the same stored trajectory.
    Tolerance: rel 1e-4 of the largest gradient component of the agent (the chained products of an
    80-step reverse pass in float32 carry ~80 * 2^-23 * |g|), plus 1e-6 absolute."""
    h, sim_d, sim, t0, acts, av, acts_d, av_d, odyn, C = _rollout(cfgid, dyn, n, B)
    Bn, T, A = sim["x"].shape
    rng = np.random.default_rng(9)
    g_rows = rng.uniform(-1, 1, (Bn, n, 5, A)).astype(np.float32)
    ga_d = torch.full((Bn, n, C, A), 7.0, device="cuda"); g0_d = torch.full((Bn, 5, A), 7.0, device="cuda")
    wm.wm_rollout_vjp(h, sim_d, t0, n, acts_d, av_d, torch.from_numpy(g_rows).cuda(), ga_d, g0_d)
    torch.cuda.synchronize()
    ref = oracle.rollout_vjp(sim, t0, n, odyn, acts, av, g_rows)
    ga, g0 = ga_d.cpu().numpy().astype(np.float64), g0_d.cpu().numpy().astype(np.float64)
    ra, r0 = ref["g_actions"].astype(np.float64), ref["g_state0"].astype(np.float64)
    scale = np.maximum(np.abs(ra).max(axis=(1, 2), keepdims=True), np.abs(r0).max(axis=1)[:, None, None, :])      # per (scenario, agent)
    assert np.all(np.abs(ga - ra) <= 1e-4 * scale + 1e-6), float(np.abs(ga - ra).max())
    assert np.all(np.abs(g0 - r0) <= 1e-4 * scale[:, 0] + 1e-6), float(np.abs(g0 - r0).max())
    # playback slots and invalid agents: exactly zero action gradient
    use_dyn = (av != 0) & (sim["valid"][:, t0:t0 + n] != 0)
    assert np.all(ga[~np.broadcast_to(use_dyn[:, :, None, :], ga.shape)] == 0.0)
    nz = int((np.abs(ra) > 0).sum())
    print("vjp cfg %d %s: %d non-zero action gradients, max |g| %.3g, max abs err %.3g" % (cfgid, dyn, nz, np.abs(ra).max(), np.abs(ga - ra).max()))
    assert nz > 0.5 * use_dyn.sum()
    wm.wm_destroy(h)


def test_step_vjp_is_the_one_step_case():
    h, sim_d, sim, t0, acts, av, acts_d, av_d, odyn, C = _rollout(1, "bicycle", 6)
    Bn, T, A = sim["x"].shape
    g_next = np.random.default_rng(2).uniform(-1, 1, (Bn, 5, A)).astype(np.float32)
    gs = torch.zeros((Bn, 5, A), device="cuda"); ga = torch.zeros((Bn, 2, A), device="cuda")
    k = 3
    wm.wm_step_vjp(h, sim_d, t0 + k, acts_d[:, k].contiguous(), av_d[:, k].contiguous(), torch.from_numpy(g_next).cuda(), gs, ga)
    torch.cuda.synchronize()
    ref = oracle.rollout_vjp(sim, t0 + k, 1, odyn, np.ascontiguousarray(acts[:, k:k + 1]), np.ascontiguousarray(av[:, k:k + 1]),
                             np.ascontiguousarray(g_next[:, None]))
    assert np.allclose(ga.cpu().numpy(), ref["g_actions"][:, 0], rtol=1e-5, atol=1e-6)
    assert np.allclose(gs.cpu().numpy(), ref["g_state0"], rtol=1e-5, atol=1e-6)
    wm.wm_destroy(h)


GRIDS = {"bicycle": ([13, 9], [-6.0, -0.3], [6.0, 0.3]), "delta_local": ([21, 21, 11], [-2.0, -0.5, -0.2], [2.0, 0.5, 0.2])}


@pytest.mark.parametrize("dyn", ["bicycle", "delta_local"])
def test_discretize_and_decode_bit_exact(dyn):
    """Same float32 inputs on both sides: bin indices, de-quantised values and the decode are bit-exact."""
    wdyn, odyn, C = DYN[dyn]
    n, lo, hi = GRIDS[dyn]
    rng = np.random.default_rng(4)
    N, A = 37, 45                                         # ragged: not a multiple of the CTA size
    act = np.stack([rng.uniform(lo[c] * 1.3, hi[c] * 1.3, (N, A)) for c in range(C)], axis=1).astype(np.float32)
    step0 = (hi[0] - lo[0]) / (n[0] - 1)
    act[0, 0, :n[0]] = (lo[0] + step0 * np.arange(n[0])).astype(np.float32)                  # grid values
    act[1, 0, :n[0] - 1] = (lo[0] + step0 * (np.arange(n[0] - 1) + 0.5)).astype(np.float32)   # bin boundaries
    valid = (rng.uniform(size=(N, A)) < 0.85).astype(np.uint8)
    h = wm.wm_create(dynamics=wdyn)
    grid = wm.action_grid(n, lo, hi)
    idx = torch.full((N, A), 99, dtype=torch.int32, device="cuda"); deq = torch.full((N, C, A), 9.0, device="cuda")
    wm.wm_discretize_actions(h, grid, torch.from_numpy(act).cuda(), idx, deq, torch.from_numpy(valid).cuda())
    back = torch.full((N, C, A), 9.0, device="cuda")
    wm.wm_actions_from_index(h, grid, idx, back)
    torch.cuda.synchronize()
    ref = oracle.discretize_actions(act, n, lo, hi, valid)
    assert np.array_equal(idx.cpu().numpy(), ref["index"])
    assert np.array_equal(deq.cpu().numpy(), ref["action"])
    assert np.array_equal(back.cpu().numpy(), oracle.actions_from_index(ref["index"], C, n, lo, hi))
    # D45: indices that are no bin of the grid (total, total + 1, INT_MAX, negative) decode to the zero action
    total = int(np.prod(n[:C]))
    odd = np.array([[total - 1, total, total + 1, 2**31 - 1, -1, -7, 0]], np.int32)
    back2 = torch.full((1, C, odd.shape[1]), 9.0, device="cuda")
    wm.wm_actions_from_index(h, grid, torch.from_numpy(odd).cuda(), back2)
    torch.cuda.synchronize()
    got = back2.cpu().numpy()
    assert np.array_equal(got, oracle.actions_from_index(odd, C, n, lo, hi))
    assert np.all(got[0, :, 1:6] == 0.0) and np.all(got[0, :, 6] == np.asarray(lo[:C], np.float32)) and np.all(got[0, :, 0] != 0.0)
    wm.wm_destroy(h)


@pytest.mark.parametrize("cfgid,dyn", [(5, "bicycle"), (2, "delta_local")])
def test_expert_actions_discrete(cfgid, dyn):
    """Discrete expert (L204) = discretised continuous inverse.  The GPU's continuous inverse differs from
    the oracle's by float32 rounding, so bins are compared outside a band around the bin boundaries
    (members counted); the de-quantised action is the grid value of the GPU's own bin, bit-exact."""
    wdyn, odyn, C = DYN[dyn]
    n, lo, hi = GRIDS[dyn]
    ns = 20
    cfg = ws.make_config(cfgid, B=16)
    log = cfg["log"]
    Bn, T, A = log["x"].shape
    h = wm.wm_create(dynamics=wdyn)
    log_d = dev(log)
    grid = wm.action_grid(n, lo, hi)
    idx = torch.zeros((Bn, ns, A), dtype=torch.int32, device="cuda"); act = torch.zeros((Bn, ns, C, A), device="cuda")
    val = torch.zeros((Bn, ns, A), dtype=torch.uint8, device="cuda")
    cont = torch.zeros((Bn, ns, C, A), device="cuda"); cval = torch.zeros((Bn, ns, A), dtype=torch.uint8, device="cuda")
    wm.wm_expert_actions_discrete(h, log_d, 10, ns, grid, idx, act, val)
    wm.wm_expert_actions(h, log_d, 10, ns, cont, cval)
    torch.cuda.synchronize()
    ref_c = oracle.expert_actions(log, 10, ns, odyn)
    assert np.array_equal(val.cpu().numpy(), ref_c["valid"])
    ref = oracle.discretize_actions(ref_c["action"], n, lo, hi, ref_c["valid"])
    # band: the oracle's continuous value within the expert tolerance of a bin boundary (or beyond the range edge bins it clamps)
    v = ref_c["valid"] != 0
    amb = np.zeros(v.shape, bool)
    tol = [2e-3, 2e-3, 2e-4] if dyn == "bicycle" else [2e-5, 2e-5, 2e-5]
    for c in range(C):
        stp = (hi[c] - lo[c]) / (n[c] - 1)
        frac = (ref_c["action"][:, :, c].astype(np.float64) - lo[c]) / stp
        amb |= np.abs(frac - np.floor(frac) - 0.5) * stp < tol[c]
    if dyn == "bicycle":                                   # Eq. 3 is ill-conditioned near standstill (D31): curvature out of the comparison there
        amb |= np.abs(ref_c["kden"]) < 0.05
    ok = v & ~amb
    gi = idx.cpu().numpy()
    assert np.array_equal(gi[ok], ref["index"][ok]), int((gi[ok] != ref["index"][ok]).sum())
    assert np.all(gi[~v] == -1)
    print("discrete expert cfg %d %s: %d transitions, %d in the band" % (cfgid, dyn, int(v.sum()), int((v & amb).sum())))
    assert (v & amb).sum() < 0.35 * v.sum()
    # de-quantised action = decode of the GPU's own index = discretisation of the GPU's own continuous inverse
    own = oracle.discretize_actions(cont.cpu().numpy(), n, lo, hi, cval.cpu().numpy())
    assert np.array_equal(gi, own["index"]) and np.array_equal(act.cpu().numpy(), own["action"])
    wm.wm_destroy(h)


@pytest.mark.parametrize("cfgid,B,k", [(1, 4, 64), (3, 2, 1000)])
def test_observe_topk_sorted_by_distance(cfgid, B, k):
    """WM_TOPK_BY_DISTANCE: indices bit-equal to the oracle's (key, index)-sorted list, features as in the index order."""
    cfg = ws.make_config(cfgid, B=B)
    log, rg = cfg["log"], cfg["roadgraph"]
    Bn, T, A = log["x"].shape
    h = wm.wm_create(topk=k, topk_order=wm.WM_TOPK_BY_DISTANCE)
    log_d, rg_d = dev(log), dev(rg)
    wm.wm_prepare(h, rg_d)
    idx = torch.zeros((Bn, A, k), dtype=torch.int32, device="cuda"); feat = torch.zeros((Bn, A, 4, k), device="cuda")
    typ = torch.zeros((Bn, A, k), dtype=torch.int32, device="cuda")
    wm.wm_observe(h, log_d, rg_d, 10, None, None, idx, feat, typ)
    torch.cuda.synchronize()
    ref = oracle.observe_topk(log, rg, 10, k, order=1)
    assert np.array_equal(idx.cpu().numpy(), ref["rg_index"])
    assert np.array_equal(typ.cpu().numpy(), ref["rg_type"])
    assert np.allclose(feat.cpu().numpy(), ref["rg_feat"], rtol=1e-5, atol=2e-4)
    wm.wm_destroy(h)
