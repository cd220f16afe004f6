"""Plumbing for the -m gpu parity tests: upload, call the C-ABI, download, compare.

Tolerances (BASELINE.json north_star; derivations in DESIGN.md "Tolerances"):
  state after one step: 1e-4 m, 1e-5 rad (velocity: 1e-3 m/s = position tolerance / dt);
  state after an 80-step free-running rollout: 1e-3 m;
  distances: rel 1e-5 plus an absolute floor of 3e-6 m (float32 rounding of the box-corner
  offsets, ~3 m * 2^-23 * a few operations);
  flags / index sets: bit-exact outside the 1e-4 m ambiguity band, band members counted.
"""
import numpy as np
import torch

import oracle
import paper_2310_08710_b200 as wm

POS_TOL, YAW_TOL, VEL_TOL = 1e-4, 1e-5, 1e-3
DIST_REL, DIST_ABS = 1e-5, 3e-6
BAND = 1e-4


def dev(d):
    return wm.to_device(d, "cuda")


def host(d):
    return {k: v.cpu().numpy() for k, v in d.items()}


def ang_diff(a, b):
    return np.abs(np.angle(np.exp(1j * (a.astype(np.float64) - b.astype(np.float64)))))


def assert_state_close(gpu_row, orc_row, pos_tol=POS_TOL, yaw_tol=YAW_TOL, vel_tol=VEL_TOL):
    """rows: dict field -> [B, A] (numpy). Validity exact; fields compared where valid."""
    assert np.array_equal(gpu_row["valid"], orc_row["valid"])
    v = orc_row["valid"] == 1
    for k, tol in (("x", pos_tol), ("y", pos_tol), ("vel_x", vel_tol), ("vel_y", vel_tol)):
        err = np.abs(gpu_row[k][v].astype(np.float64) - orc_row[k][v])
        assert err.max(initial=0) <= tol, (k, err.max())
    assert ang_diff(gpu_row["yaw"][v], orc_row["yaw"][v]).max(initial=0) <= yaw_tol
    assert np.array_equal(gpu_row["length"][v], orc_row["length"][v])
    assert np.array_equal(gpu_row["width"][v], orc_row["width"][v])


def row_of(tr, t):
    return {k: v[:, t] for k, v in tr.items()}


def gpu_offroad(h, sim_d, t):
    B, T, A = sim_d["x"].shape
    sd = torch.full((B, A), 7.0, device="cuda"); cd = torch.full((B, 4, A), 7.0, device="cuda")
    fl = torch.full((B, A), 9, dtype=torch.uint8, device="cuda")
    wm.wm_metrics_offroad(h, sim_d, t, sd, cd, fl)
    torch.cuda.synchronize()
    return sd.cpu().numpy(), cd.cpu().numpy(), fl.cpu().numpy()


def compare_offroad(sd, cd, fl, orc, valid):
    """GPU (sd [B,A], cd [B,4,A], fl [B,A]) against oracle.offroad(...) output. Returns stats."""
    v = valid == 1
    # invalid agents: zeros (D10)
    assert np.all(sd[~v] == 0) and np.all(fl[~v] == 0) and np.all(cd[np.broadcast_to(~v[:, None, :], cd.shape)] == 0)
    amb = orc["ambig"] == 1
    vc = np.broadcast_to(v[:, None, :], cd.shape)
    ok = vc & ~amb
    ref = orc["corner_dist"].astype(np.float64)
    err = np.abs(cd.astype(np.float64) - ref)
    tol = DIST_REL * np.abs(ref) + DIST_ABS
    bad = ok & (err > tol)
    assert not bad.any(), ("corner distance mismatch", int(bad.sum()), float(err[bad].max()), np.argwhere(bad)[:5])
    # ambiguous corners: the magnitude must still agree (only the sign / winner may differ)
    ambv = vc & amb
    errm = np.abs(np.abs(cd.astype(np.float64)) - np.abs(ref))
    assert (errm[ambv] <= tol[ambv] + BAND).all()
    clean = v & ~amb.any(axis=1)
    assert np.array_equal(fl[clean], orc["flag"][clean]), "offroad flag mismatch outside the band"
    errs = np.abs(sd.astype(np.float64)[clean] - orc["signed_dist"].astype(np.float64)[clean])
    assert (errs <= DIST_REL * np.abs(orc["signed_dist"][clean]) + DIST_ABS).all()
    # a non-ambiguous positive corner forces the flag even if another corner is ambiguous
    sure_pos = (ok & (ref > 0)).any(axis=1)
    assert np.all(fl[v & sure_pos] == 1)
    return dict(corners=int(vc.sum()), ambiguous=int(ambv.sum()), agents_clean=int(clean.sum()))


def gpu_overlap(h, sim_d, t):
    B, T, A = sim_d["x"].shape
    W = (A + 31) // 32
    bits = torch.full((B, A, W), -1, dtype=torch.int32, device="cuda")
    fl = torch.full((B, A), 9, dtype=torch.uint8, device="cuda")
    wm.wm_metrics_overlap(h, sim_d, t, bits, fl)
    torch.cuda.synchronize()
    bits = bits.cpu().numpy().view(np.uint32)
    pair = ((bits[..., None] >> np.arange(32, dtype=np.uint32)) & 1).reshape(B, A, W * 32)[:, :, :A].astype(np.uint8)
    return pair, fl.cpu().numpy()


def compare_overlap(pair, fl, orc, valid):
    gap = orc["gap"]
    amb = np.abs(gap) < BAND
    ok = ~amb
    assert np.array_equal(pair[ok], orc["pair"][ok]), "overlap pair mismatch outside the band"
    assert np.array_equal(pair, np.transpose(pair, (0, 2, 1)))
    assert np.array_equal(fl, pair.max(axis=2)), "flag must be the row OR of the pair bits"
    clean = ~amb.any(axis=2)
    assert np.array_equal(fl[clean], orc["flag"][clean])
    inv = valid == 0
    assert pair[inv].sum() == 0 and fl[inv].sum() == 0
    return dict(pairs=int(ok.sum()), ambiguous=int(amb.sum()), overlap_frac=float(orc["pair"].mean()))
