"""Float64 restatements, in plain numpy and straight from the definitions in include/wm.h / DESIGN.md, of the two
places where a float32 value decides an INDEX and the oracle deliberately follows the kernel's float32 operations
(route progress D33, IDM lead D39).  They share nothing with oracle/ or the CUDA path.  The CPU suite pins the
oracle with them; the GPU suite checks the kernels' choices with them.  Both compare only where the decision is
clear by more than a band of 1e-4 m and count the rest."""
import numpy as np


def route_ratio_in_double(log, sim, t, paths, band=1e-4):
    """L96 / D33-D35 in float64 with numpy, written from the definition: closest valid path POINT to the simulated
    position at t and to the first / last valid logged position.  Returns (ratio, decided): decided = every one of
    the three closest-point choices beats by more than `band` metres every runner-up with another arc length (a parked
    agent's coincident path points all carry the same one), the agent is valid and d_q != d_p."""
    B, T, A = log["x"].shape
    ratio = np.zeros((B, A)); decided = np.zeros((B, A), bool)
    for b in range(B):
        for a in range(A):
            pv = paths["valid"][b, a] == 1
            lv = np.nonzero(log["valid"][b, :, a] == 1)[0]
            if sim["valid"][b, t, a] != 1 or not pv.any() or lv.size == 0:
                continue
            px, py, arc = paths["x"][b, a].astype(np.float64), paths["y"][b, a].astype(np.float64), paths["arc_len"][b, a].astype(np.float64)
            pick, sure = [], True
            for qx, qy in ((sim["x"][b, t, a], sim["y"][b, t, a]), (log["x"][b, lv[0], a], log["y"][b, lv[0], a]), (log["x"][b, lv[-1], a], log["y"][b, lv[-1], a])):
                d = np.where(pv, np.hypot(px - float(qx), py - float(qy)), np.inf)
                i = int(np.argmin(d))
                near = d <= d[i] + band                            # runners-up the float32 key could prefer ...
                sure &= bool(np.all(arc[near] == arc[i]))          # ... matter only if they sit elsewhere along the path
                pick.append(i)
            dx, dp, dq = arc[pick[0]], arc[pick[1]], arc[pick[2]]
            if dq != dp:
                ratio[b, a] = (dx - dp) / (dq - dp); decided[b, a] = sure
    return ratio, decided


def idm_lead_in_double(sim, t, paths, idm, band=1e-4):
    """The lead object of D38 / D39 in float64 with numpy, written from the definition (include/wm.h wm_idm_step):
    project every agent on agent i's path (nearest path segment between index-consecutive valid points, arc length
    of the projection), keep those ahead (sigma_j > sigma_i) within (W_i + W_j) / 2 of the path, take the smallest
    gap sigma_j - sigma_i - (L_i + L_j) / 2.  Returns (lead [B][A], decided [B][A]): decided = no comparison that
    picks the lead was closer than `band` metres (ahead or not, inside the corridor or not, best gap against the
    next, nearest segment against another one elsewhere along the path); only there must a float32 implementation
    agree."""
    B, T, A = sim["x"].shape
    lead = np.full((B, A), -1, np.int64); decided = np.zeros((B, A), bool)
    for b in range(B):
        X, Y = sim["x"][b, t].astype(np.float64), sim["y"][b, t].astype(np.float64)
        L, W, V = sim["length"][b, t].astype(np.float64), sim["width"][b, t].astype(np.float64), sim["valid"][b, t] == 1
        for i in range(A):
            if not idm[b, i] or not V[i]:
                decided[b, i] = True
                continue
            pv = paths["valid"][b, i] == 1
            seg = np.nonzero(pv[:-1] & pv[1:])[0]
            if seg.size == 0:
                decided[b, i] = True
                continue
            px, py, arc = paths["x"][b, i].astype(np.float64), paths["y"][b, i].astype(np.float64), paths["arc_len"][b, i].astype(np.float64)
            ex, ey = px[seg + 1] - px[seg], py[seg + 1] - py[seg]
            ee = ex * ex + ey * ey
            wx, wy = X[:, None] - px[seg][None, :], Y[:, None] - py[seg][None, :]                 # [A][S]
            u = np.where(ee > 0, np.clip((wx * ex + wy * ey) / np.where(ee > 0, ee, 1.0), 0.0, 1.0), 0.0)
            d = np.hypot(wx - u * ex, wy - u * ey)
            sg = arc[seg][None, :] + u * (arc[seg + 1] - arc[seg])[None, :]
            k = np.argmin(d, axis=1)
            ar = np.arange(A)
            dist, sigma = d[ar, k], sg[ar, k]
            # another segment as near (within band) that puts the projection elsewhere along the path
            shaky = ((d <= dist[:, None] + band) & (np.abs(sg - sigma[:, None]) > 1e-3)).any(axis=1)
            lat = 0.5 * (W[i] + W)
            gap = sigma - sigma[i] - 0.5 * (L[i] + L)
            other = V & (ar != i)
            sure_in = other & ~shaky & (sigma > sigma[i] + band) & (dist < lat - band)
            # (whichever of several equally near segments is taken, an agent farther than the corridor stays outside it)
            sure_out = ~other | (dist > lat + 2 * band) | (~shaky & (sigma < sigma[i] - band))
            maybe = ~sure_in & ~sure_out
            if shaky[i]:
                continue
            if not sure_in.any():
                decided[b, i] = not maybe.any()
                continue
            g = np.where(sure_in, gap, np.inf)
            j = int(np.argmin(g))
            rest = np.delete(g, j)
            clear = (rest.size == 0 or rest.min() - g[j] > 2 * band) and not (maybe & (gap <= g[j] + 2 * band)).any()
            lead[b, i] = j; decided[b, i] = clear
    return lead, decided
