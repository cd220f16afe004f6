"""Pins for the oracle's pairwise oriented-box overlap (O3)."""
import math
import os

import numpy as np
import pytest

import oracle
from util import boxes_traj, rigid

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "overlap_hand_cases.txt")


def _cases():
    out = []
    for line in open(GOLDEN):
        line = line.split("#")[0].strip()
        if not line:
            continue
        v = [float(q) for q in line.split()]
        out.append((v[0:5], v[5:10], int(v[10])))
    return out


# P6: hand cases
@pytest.mark.parametrize("b1,b2,expected", _cases())
def test_overlap_hand_cases(b1, b2, expected):
    boxes = [(b[0], b[1], math.radians(b[2]), b[3], b[4]) for b in (b1, b2)]
    out = oracle.overlap(boxes_traj(boxes), 0)
    assert out["pair"][0, 0, 1] == expected and out["pair"][0, 1, 0] == expected
    assert out["flag"][0, 0] == expected and out["flag"][0, 1] == expected
    assert out["pair"][0, 0, 0] == 0 and out["pair"][0, 1, 1] == 0


def test_gap_value_on_axis_aligned_boxes():
    # the separating gap equals the face-to-face distance for axis-aligned boxes
    out = oracle.overlap(boxes_traj([(0, 0, 0, 2, 2), (2.01, 0, 0, 2, 2), (0, 5, 0, 2, 2)]), 0)
    assert out["gap"][0, 0, 1] == pytest.approx(0.01, abs=1e-6)
    assert out["gap"][0, 0, 2] == pytest.approx(3.0, abs=1e-6)
    assert out["gap"][0, 1, 2] == pytest.approx(3.0, abs=1e-6)   # max over axes, not Euclidean


# ---- P7: brute force by polygon clipping (Sutherland-Hodgman), independent of SAT ----
def _corners(x, y, yaw, L, W):
    c, s = math.cos(yaw), math.sin(yaw)
    pts = []
    for sl, sw in ((1, 1), (-1, 1), (-1, -1), (1, -1)):     # counter-clockwise
        pts.append((x + sl * L / 2 * c - sw * W / 2 * s, y + sl * L / 2 * s + sw * W / 2 * c))
    return pts


def _clip(subject, clipper):
    out = subject
    n = len(clipper)
    for i in range(n):
        a, b = clipper[i], clipper[(i + 1) % n]
        inp, out = out, []
        if not inp:
            break

        def inside(p):
            return (b[0] - a[0]) * (p[1] - a[1]) - (b[1] - a[1]) * (p[0] - a[0]) >= 0

        def inter(p, q):
            d1 = (b[0] - a[0], b[1] - a[1]); d2 = (q[0] - p[0], q[1] - p[1])
            den = d1[0] * d2[1] - d1[1] * d2[0]
            tt = ((p[0] - a[0]) * d2[1] - (p[1] - a[1]) * d2[0]) / den
            return (a[0] + tt * d1[0], a[1] + tt * d1[1])

        for k in range(len(inp)):
            p, q = inp[k - 1], inp[k]
            if inside(q):
                if not inside(p):
                    out.append(inter(p, q))
                out.append(q)
            elif inside(p):
                out.append(inter(p, q))
    return out


def _area(poly):
    return 0.5 * abs(sum(poly[i - 1][0] * poly[i][1] - poly[i][0] * poly[i - 1][1] for i in range(len(poly))))


def test_overlap_matches_polygon_clipping_bruteforce():
    n_checked = n_band = n_overlap = 0
    for seed in range(250):
        rng = np.random.default_rng(seed)
        A = 12
        boxes = [(rng.uniform(0, 14), rng.uniform(0, 14), rng.uniform(-math.pi, math.pi),
                  rng.uniform(0.5, 5.5), rng.uniform(0.5, 2.2)) for _ in range(A)]
        tr = boxes_traj(boxes)
        out = oracle.overlap(tr, 0)
        # use exactly the float32 values the oracle saw
        fb = [tuple(float(tr[k][0, 0, a]) for k in ("x", "y", "yaw", "length", "width")) for a in range(A)]
        for i in range(A):
            for j in range(i + 1, A):
                if abs(out["gap"][0, i, j]) < 1e-4:        # band-excluded (P15)
                    n_band += 1
                    continue
                inter = _clip(_corners(*fb[i]), _corners(*fb[j]))
                brute = len(inter) >= 3 and _area(inter) > 1e-9
                assert bool(out["pair"][0, i, j]) == brute, (seed, i, j, out["gap"][0, i, j])
                n_checked += 1
                n_overlap += brute
    assert n_checked > 15000 and n_overlap > 500


# P8: invariants
def test_overlap_invariants():
    import wm_scenarios as ws
    cfg = ws.make_config(4, B=2)
    tr = cfg["log"]
    tr["valid"][0, 0, 5:40:3] = 0            # punch some invalid agents
    for k in ("x", "y", "yaw", "length", "width"):
        tr[k][0, 0, 5:40:3] = np.nan
    out = oracle.overlap(tr, 0)
    pair, gap = out["pair"], out["gap"]
    assert np.array_equal(pair, np.transpose(pair, (0, 2, 1)))                 # symmetric
    assert np.all(pair[:, np.arange(512), np.arange(512)] == 0)                # diagonal
    inv = tr["valid"][:, 0] == 0
    assert pair[inv].sum() == 0 and np.transpose(pair, (0, 2, 1))[inv].sum() == 0
    assert np.array_equal(out["flag"], pair.max(axis=2))                       # flag = row OR
    frac = pair[1].sum() / (512 * 511)
    assert 0.002 < frac < 0.03        # crowded lot: a car only reaches its ~8 neighbours
    # rigid transform + yaw->yaw+pi leave every pair outside the band unchanged
    tr2, _ = rigid(tr, None, 0.83, 40.0, -25.0)
    tr2["yaw"][:, :, ::2] += np.float32(math.pi)
    out2 = oracle.overlap(tr2, 0)
    stable = np.abs(gap) > 1e-3
    assert np.array_equal(out2["pair"][stable], pair[stable])
    assert np.nanmax(np.abs(out2["gap"][stable & np.isfinite(gap)] - gap[stable & np.isfinite(gap)])) < 2e-4
