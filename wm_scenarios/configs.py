"""The five BASELINE.json configs as seeded synthetic scenario batches (numpy, host).

Layouts (the C-ABI's, include/wm.h): trajectories ``[B][T][A]`` time-major SoA, roadgraph
``[B][R]`` SoA, actions ``[B][n_steps][C][A]``.  All floats are generated in float64 and
rounded once to float32.  Nothing here evaluates the simulator's equations; the recipe is
described in DESIGN.md ("Input recipe").
"""
import numpy as np

from .rng import uniform, randint, MASTER_SEED

TYPE_LANE = 1
TYPE_ROAD_EDGE = 2

DT = 0.1
HISTORY = 11

# name -> (B, A, R, T)
CONFIG_SHAPES = {
    1: dict(B=4, A=32, R=2000, T=91),
    2: dict(B=512, A=128, R=30000, T=91),
    3: dict(B=256, A=128, R=30000, T=91),
    4: dict(B=64, A=512, R=5000, T=1),
    5: dict(B=4096, A=128, R=20000, T=91),
}

# random streams (names of the quantities drawn)
(S_SLOT, S_SLOT2, S_JIT, S_ABLOCK, S_ALANE, S_APOINT, S_ATYPE, S_ALEN, S_AWID, S_ASPEED,
 S_AVALID, S_AACC, S_AKAPPA, S_ACT0, S_ACT1, S_ACT2, S_LATE, S_LATE_T, S_LANEKIND, S_LANEPOS,
 S_LANEYAW, S_LANERAD, S_YAW, S_JITX, S_JITY) = range(25)


# --------------------------------------------------------------------------------------
# logged trajectories: exact arcs (closed form; data recipe, not the simulator's update)
# --------------------------------------------------------------------------------------
def arc_trajectory(x0, y0, yaw0, v0, acc, kappa, vmax, T, dt=DT):
    """Constant-acceleration (speed clipped to [0, vmax]), constant-curvature arc.

    Inputs broadcastable arrays [...]; returns x, y, yaw, vx, vy of shape [..., T] (float64).
    Arclength s(t) is the exact integral of the clipped speed; the position is the exact
    chord of a circular arc: p = p0 + s*sinc(kappa*s/2) * (cos, sin)(yaw0 + kappa*s/2).
    """
    t = np.arange(T, dtype=np.float64) * dt
    x0, y0, yaw0, v0, acc, kappa, vmax = [np.asarray(q, dtype=np.float64)[..., None]
                                          for q in (x0, y0, yaw0, v0, acc, kappa, vmax)]
    with np.errstate(divide="ignore", invalid="ignore"):
        # time at which the speed hits a clip (0 for braking, vmax for accelerating)
        t_clip = np.where(acc > 0, (vmax - v0) / acc, np.where(acc < 0, v0 / (-acc), np.inf))
    t_clip = np.where(np.isfinite(t_clip), np.maximum(t_clip, 0.0), np.inf)
    te = np.minimum(t, t_clip)
    v_clip = np.where(acc > 0, vmax, 0.0)
    s = v0 * te + 0.5 * acc * te * te + np.where(t > t_clip, v_clip * (t - np.minimum(t_clip, t)), 0.0)
    v = np.where(t > t_clip, v_clip, v0 + acc * te)
    half = 0.5 * kappa * s
    chord = s * np.sinc(half / np.pi)
    yaw = yaw0 + kappa * s
    x = x0 + chord * np.cos(yaw0 + half)
    y = y0 + chord * np.sin(yaw0 + half)
    return x, y, yaw, v * np.cos(yaw), v * np.sin(yaw)


def _empty_traj(B, T, A):
    tr = {k: np.zeros((B, T, A), dtype=np.float32)
          for k in ("x", "y", "yaw", "vel_x", "vel_y", "length", "width")}
    tr["valid"] = np.zeros((B, T, A), dtype=np.uint8)
    return tr


def _fill_traj(tr, sl, x, y, yaw, vx, vy, length, width, valid_ta, poison):
    """x.. are [b, A, T] float64; valid_ta is [b, A, T] bool. Writes time-major [b, T, A]."""
    bad = ~valid_ta
    for k, v in (("x", x), ("y", y), ("yaw", yaw), ("vel_x", vx), ("vel_y", vy),
                 ("length", np.broadcast_to(length[..., None], x.shape)),
                 ("width", np.broadcast_to(width[..., None], x.shape))):
        v = np.array(v, dtype=np.float64, copy=True)
        v[bad] = np.nan if poison else 0.0
        tr[k][sl] = np.transpose(v, (0, 2, 1)).astype(np.float32)
    tr["valid"][sl] = np.transpose(valid_ta, (0, 2, 1)).astype(np.uint8)


# --------------------------------------------------------------------------------------
# street-block roadgraph (configs 2, 3, 5)
# --------------------------------------------------------------------------------------
def _slot_tables():
    main, half = [], []
    for j in range(5):
        for i in range(4):
            main.append((50.0 * i + 25.0, 50.0 * j, 1.0, 0.0))    # horizontal street piece
            main.append((50.0 * j, 50.0 * i + 25.0, 0.0, 1.0))    # vertical street piece
    for j in range(4):
        for i in range(4):
            half.append((50.0 * i + 25.0, 50.0 * j + 25.0, 1.0, 0.0))
            half.append((50.0 * j + 25.0, 50.0 * i + 25.0, 0.0, 1.0))
    return np.array(main), np.array(half)  # [40,4], [32,4]


_MAIN_SLOTS, _HALF_SLOTS = _slot_tables()
# spatial order across the street: edge, 2 lanes (+dir), 2 lanes (-dir), edge
_POLY_OFFSET = np.array([-7.0, -5.25, -1.75, 1.75, 5.25, 7.0])
_POLY_SIGN = np.array([1.0, 1.0, 1.0, -1.0, -1.0, -1.0])   # travel / point-order direction
_POLY_TYPE = np.array([TYPE_ROAD_EDGE, TYPE_LANE, TYPE_LANE, TYPE_LANE, TYPE_LANE, TYPE_ROAD_EDGE])
_LANE_POLYS = np.array([1, 2, 3, 4])
_PTS = 100
_SPACING = 0.5


def _street_blocks(seed, b, n_blocks):
    """Per scenario: block centres [b, nb, 2] (jittered) and street directions [b, nb, 2]."""
    k1 = uniform(seed, b, S_SLOT, (40,))
    k2 = uniform(seed, b, S_SLOT2, (32,))
    p1 = np.argsort(k1, axis=-1, kind="stable")
    p2 = np.argsort(k2, axis=-1, kind="stable")
    n1 = min(n_blocks, 40)
    slots = _MAIN_SLOTS[p1[:, :n1]]
    if n_blocks > 40:
        n2 = n_blocks - 40
        if n2 > 32:
            raise ValueError("street-block generator supports at most 72 blocks (R <= 43200)")
        slots = np.concatenate([slots, _HALF_SLOTS[p2[:, :n2]]], axis=1)
    jit = uniform(seed, b, S_JIT, (n_blocks, 2), -2.0, 2.0)
    return slots[..., 0:2] + jit, slots[..., 2:4]


def _street_roadgraph(seed, b, R):
    nb = R // 600
    Bn = len(b)
    ctr, d = _street_blocks(seed, b, nb)                       # [b, nb, 2]
    nrm = np.stack([-d[..., 1], d[..., 0]], axis=-1)           # left normal of the street axis
    s = (-24.75 + _SPACING * np.arange(_PTS))                  # along-street coordinate
    # [b, nb, 6, 100, 2]
    sgn = _POLY_SIGN[None, None, :, None, None]
    along = (sgn * s[None, None, None, :, None]) * d[:, :, None, None, :]
    lateral = _POLY_OFFSET[None, None, :, None, None] * nrm[:, :, None, None, :]
    pts = ctr[:, :, None, None, :] + along + lateral
    dirs = np.broadcast_to(sgn * d[:, :, None, None, :], pts.shape)
    rg = {
        "x": np.zeros((Bn, R), np.float32), "y": np.zeros((Bn, R), np.float32),
        "dir_x": np.ones((Bn, R), np.float32), "dir_y": np.zeros((Bn, R), np.float32),
        "type": np.zeros((Bn, R), np.int32), "id": np.full((Bn, R), -1, np.int32),
        "valid": np.zeros((Bn, R), np.uint8),
    }
    n = nb * 600
    rg["x"][:, :n] = pts[..., 0].reshape(Bn, n)
    rg["y"][:, :n] = pts[..., 1].reshape(Bn, n)
    rg["dir_x"][:, :n] = dirs[..., 0].reshape(Bn, n)
    rg["dir_y"][:, :n] = dirs[..., 1].reshape(Bn, n)
    rg["type"][:, :n] = np.broadcast_to(_POLY_TYPE[None, None, :, None], (Bn, nb, 6, _PTS)).reshape(Bn, n)
    rg["id"][:, :n] = np.broadcast_to(
        (np.arange(nb)[:, None] * 6 + np.arange(6)[None, :])[None, :, :, None], (Bn, nb, 6, _PTS)).reshape(Bn, n)
    rg["valid"][:, :n] = 1
    return rg, ctr, d, nrm


def make_street_scenarios(seed, b_ids, A, R, T, invalid_frac=0.15, late_frac=0.05,
                          poison_invalid=True, chunk=256):
    """Configs 2/3/5 scenario data for scenario ids ``b_ids`` (int array)."""
    b_ids = np.asarray(b_ids, dtype=np.int64)
    Bn = len(b_ids)
    nb = R // 600
    log = _empty_traj(Bn, T, A)
    rgs = None
    for c0 in range(0, Bn, chunk):
        sl = slice(c0, min(c0 + chunk, Bn))
        b = b_ids[sl]
        rg, ctr, d, nrm = _street_roadgraph(seed, b, R)
        if rgs is None:
            rgs = {k: np.zeros((Bn,) + v.shape[1:], v.dtype) for k, v in rg.items()}
        for k, v in rg.items():
            rgs[k][sl] = v
        # ---- agents on random lane points ----
        blk = randint(seed, b, S_ABLOCK, (A,), nb)
        lane = randint(seed, b, S_ALANE, (A,), 4)
        pt = randint(seed, b, S_APOINT, (A,), _PTS)
        poly = _LANE_POLYS[lane]
        bi = np.arange(len(b))[:, None]
        dd = d[bi, blk] * _POLY_SIGN[poly][..., None]          # travel direction [b, A, 2]
        pos = (ctr[bi, blk] + (_POLY_SIGN[poly] * (-24.75 + _SPACING * pt))[..., None] * d[bi, blk]
               + _POLY_OFFSET[poly][..., None] * nrm[bi, blk])
        yaw0 = np.arctan2(dd[..., 1], dd[..., 0])
        ut = uniform(seed, b, S_ATYPE, (A,))
        kind = np.where(ut < 0.7, 0, np.where(ut < 0.9, 1, 2))   # vehicle / pedestrian / cyclist
        ul = uniform(seed, b, S_ALEN, (A,))
        uw = uniform(seed, b, S_AWID, (A,))
        length = np.choose(kind, [4.0 + 1.5 * ul, 0.5 + 0.5 * ul, 1.5 + 0.5 * ul])
        width = np.choose(kind, [1.8 + 0.4 * uw, 0.5 + 0.5 * ul, 0.6 + 0.2 * uw])  # pedestrians square
        vmax = np.choose(kind, [15.0, 2.0, 8.0])
        v0 = uniform(seed, b, S_ASPEED, (A,)) * vmax
        acc = uniform(seed, b, S_AACC, (A,), -3.0, 3.0)
        kap = uniform(seed, b, S_AKAPPA, (A,), -0.1, 0.1)
        x, y, yaw, vx, vy = arc_trajectory(pos[..., 0], pos[..., 1], yaw0, v0, acc, kap, vmax, T)
        valid_a = uniform(seed, b, S_AVALID, (A,)) >= invalid_frac
        late = uniform(seed, b, S_LATE, (A,)) < late_frac
        t_on = np.where(late, randint(seed, b, S_LATE_T, (A,), 55) + 5, 0)
        valid_ta = valid_a[..., None] & (np.arange(T)[None, None, :] >= t_on[..., None])
        _fill_traj(log, sl, x, y, yaw, vx, vy, length, width, valid_ta, poison_invalid)
    return log, rgs


# --------------------------------------------------------------------------------------
# config 1: 20 short straight / arc lanes
# --------------------------------------------------------------------------------------
def _lane_polyline(p0, yaw0, kappa, s):
    """Points of a constant-curvature centreline at arclengths s: [..., n, 2] and headings."""
    half = 0.5 * kappa[..., None] * s
    chord = s * np.sinc(half / np.pi)
    yaw = yaw0[..., None] + kappa[..., None] * s
    pts = p0[..., None, :] + chord[..., None] * np.stack(
        [np.cos(yaw0[..., None] + half), np.sin(yaw0[..., None] + half)], axis=-1)
    return pts, yaw


def _dirs_from_points(pts):
    """dir of point i = unit(p[i+1]-p[i]); the last point copies its predecessor."""
    dv = pts[..., 1:, :] - pts[..., :-1, :]
    dv = dv / np.linalg.norm(dv, axis=-1, keepdims=True)
    return np.concatenate([dv, dv[..., -1:, :]], axis=-2)


def make_config1(seed=None, b_ids=None, poison_invalid=True, n_steps=80):
    shp = CONFIG_SHAPES[1]
    seed = MASTER_SEED + 1 if seed is None else seed
    b = np.arange(shp["B"]) if b_ids is None else np.asarray(b_ids, dtype=np.int64)
    Bn, A, R, T = len(b), shp["A"], shp["R"], shp["T"]
    NL = 20
    arc = uniform(seed, b, S_LANEKIND, (NL,)) < 0.5
    rad = uniform(seed, b, S_LANERAD, (NL,), 15.0, 60.0)
    sense = np.where(uniform(seed, b, S_SLOT, (NL,)) < 0.5, -1.0, 1.0)
    kappa = np.where(arc, sense / rad, 0.0)
    p0 = uniform(seed, b, S_LANEPOS, (NL, 2), 10.0, 90.0)
    yaw0 = uniform(seed, b, S_LANEYAW, (NL,), -np.pi, np.pi)
    s_c = _SPACING * np.arange(34)
    s_e = _SPACING * np.arange(33)
    ctr, _ = _lane_polyline(p0, yaw0, kappa, s_c)                   # [b, NL, 34, 2]
    ce, yaw_e = _lane_polyline(p0, yaw0, kappa, s_e)                # [b, NL, 33, 2]
    nrm = np.stack([-np.sin(yaw_e), np.cos(yaw_e)], axis=-1)        # left normal
    right = ce - 1.75 * nrm                                         # runs with the lane
    left = (ce + 1.75 * nrm)[..., ::-1, :]                          # runs against it
    polys = [(ctr, TYPE_LANE), (right, TYPE_ROAD_EDGE), (left, TYPE_ROAD_EDGE)]
    rg = {k: [] for k in ("x", "y", "dir_x", "dir_y", "type", "id")}
    for li in range(NL):
        for pi, (pts, typ) in enumerate(polys):
            p = pts[:, li]
            dv = _dirs_from_points(p)
            n = p.shape[1]
            rg["x"].append(p[..., 0]); rg["y"].append(p[..., 1])
            rg["dir_x"].append(dv[..., 0]); rg["dir_y"].append(dv[..., 1])
            rg["type"].append(np.full((Bn, n), typ)); rg["id"].append(np.full((Bn, n), li * 3 + pi))
    out = {}
    for k in ("x", "y", "dir_x", "dir_y"):
        out[k] = np.concatenate(rg[k], axis=1).astype(np.float32)
    out["type"] = np.concatenate(rg["type"], axis=1).astype(np.int32)
    out["id"] = np.concatenate(rg["id"], axis=1).astype(np.int32)
    assert out["x"].shape[1] == R
    out["valid"] = np.ones((Bn, R), np.uint8)
    # ---- agents ----
    lane = randint(seed, b, S_ALANE, (A,), NL)
    s_a = uniform(seed, b, S_APOINT, (A,), 0.0, 16.5)
    bi = np.arange(Bn)[:, None]
    pa, ya = _lane_polyline(p0[bi, lane], yaw0[bi, lane], kappa[bi, lane], s_a[..., None])
    pa, ya = pa[..., 0, :], ya[..., 0]
    v0 = uniform(seed, b, S_ASPEED, (A,), 0.0, 15.0)
    length = uniform(seed, b, S_ALEN, (A,), 4.0, 5.5)
    width = uniform(seed, b, S_AWID, (A,), 1.8, 2.2)
    acc = uniform(seed, b, S_AACC, (A,), -3.0, 3.0)
    kap = uniform(seed, b, S_AKAPPA, (A,), -0.1, 0.1)
    x, y, yaw, vx, vy = arc_trajectory(pa[..., 0], pa[..., 1], ya, v0, acc, kap, np.full_like(v0, 60.0), T)
    valid_a = uniform(seed, b, S_AVALID, (A,)) >= 0.10
    log = _empty_traj(Bn, T, A)
    _fill_traj(log, slice(0, Bn), x, y, yaw, vx, vy, length, width,
               np.broadcast_to(valid_a[..., None], x.shape).copy(), poison_invalid)
    act, act_valid = bicycle_actions(seed, b, A, n_steps, log["valid"][:, HISTORY - 1, :])
    return dict(config=1, seed=seed, b_ids=b, log=log, roadgraph=out, actions=act,
                action_valid=act_valid, dynamics="bicycle", n_steps=n_steps, t0=HISTORY - 1)


def bicycle_actions(seed, b, A, n_steps, valid_t0):
    """i.i.d. (accel U(-3,3), curvature U(-0.1,0.1)) per (b, step, agent): [B][n_steps][2][A]."""
    a = uniform(seed, b, S_ACT0, (n_steps, A), -3.0, 3.0)
    k = uniform(seed, b, S_ACT1, (n_steps, A), -0.1, 0.1)
    act = np.stack([a, k], axis=2).astype(np.float32)
    act_valid = np.broadcast_to(valid_t0[:, None, :], (len(b), n_steps, A)).astype(np.uint8).copy()
    return act, act_valid


def delta_actions(seed, b, A, valid_t0):
    """(dx, dy U(-0.5,0.5) m; dyaw U(-0.1,0.1) rad) for one step: [B][1][3][A]."""
    dx = uniform(seed, b, S_ACT0, (1, A), -0.5, 0.5)
    dy = uniform(seed, b, S_ACT1, (1, A), -0.5, 0.5)
    dw = uniform(seed, b, S_ACT2, (1, A), -0.1, 0.1)
    act = np.stack([dx, dy, dw], axis=2).astype(np.float32)
    return act, valid_t0[:, None, :].astype(np.uint8).copy()


# --------------------------------------------------------------------------------------
# config 4: crowded lot
# --------------------------------------------------------------------------------------
def make_config4(seed=None, b_ids=None, B=None, poison_invalid=True):
    shp = CONFIG_SHAPES[4]
    seed = MASTER_SEED + 4 if seed is None else seed
    b = np.arange(shp["B"] if B is None else B) if b_ids is None else np.asarray(b_ids, dtype=np.int64)
    Bn, A, R, T = len(b), shp["A"], shp["R"], shp["T"]
    gx, gy = np.meshgrid(np.arange(16), np.arange(32), indexing="ij")
    cx = (gx.reshape(-1) + 0.5) * 3.0
    cy = (gy.reshape(-1) + 0.5) * 6.0
    x = cx[None, :] + uniform(seed, b, S_JITX, (A,), -0.5, 0.5)
    y = cy[None, :] + uniform(seed, b, S_JITY, (A,), -0.5, 0.5)
    yaw = uniform(seed, b, S_YAW, (A,), -np.pi, np.pi)
    length = uniform(seed, b, S_ALEN, (A,), 4.0, 5.5)
    width = uniform(seed, b, S_AWID, (A,), 1.8, 2.2)
    valid = np.ones((Bn, A, 1), bool)
    log = _empty_traj(Bn, T, A)
    z = np.zeros((Bn, A, 1))
    _fill_traj(log, slice(0, Bn), x[..., None], y[..., None], yaw[..., None], z, z, length, width,
               valid, poison_invalid)
    # lot boundary: rectangle [-1,49] x [-1,193] (1 m margin, so border cars can poke out), counter-clockwise (interior on the left),
    # one open polyline of R points at perimeter/R spacing (last gap stays open).
    x0, x1, y0, y1 = -1.0, 49.0, -1.0, 193.0
    w, h = x1 - x0, y1 - y0
    per = 2 * (w + h)
    s = np.arange(R) * (per / R)
    px = np.where(s < w, x0 + s, np.where(s < w + h, x1, np.where(s < 2 * w + h, x1 - (s - w - h), x0)))
    py = np.where(s < w, y0, np.where(s < w + h, y0 + (s - w), np.where(s < 2 * w + h, y1, y1 - (s - 2 * w - h))))
    pts = np.stack([px, py], axis=-1)
    dv = _dirs_from_points(pts)
    rg = {
        "x": np.broadcast_to(px.astype(np.float32), (Bn, R)).copy(),
        "y": np.broadcast_to(py.astype(np.float32), (Bn, R)).copy(),
        "dir_x": np.broadcast_to(dv[:, 0].astype(np.float32), (Bn, R)).copy(),
        "dir_y": np.broadcast_to(dv[:, 1].astype(np.float32), (Bn, R)).copy(),
        "type": np.full((Bn, R), TYPE_ROAD_EDGE, np.int32),
        "id": np.zeros((Bn, R), np.int32),
        "valid": np.ones((Bn, R), np.uint8),
    }
    return dict(config=4, seed=seed, b_ids=b, log=log, roadgraph=rg, actions=None,
                action_valid=None, dynamics=None, n_steps=0, t0=0)


# --------------------------------------------------------------------------------------
def make_config(cfg, B=None, b_ids=None, seed=None, R=None, A=None, T=None, n_steps=None,
                poison_invalid=True):
    """Scenario batch for BASELINE.json config ``cfg`` (1..5).

    ``B``/``b_ids`` select a sub-batch (scenario b is the same in any batch); ``R``, ``A``,
    ``T`` override the config's shape for shrunken test cases.
    """
    if cfg == 1:
        d = make_config1(seed, b_ids if b_ids is not None else (np.arange(B) if B else None),
                         poison_invalid, n_steps=80 if n_steps is None else n_steps)
        return d
    if cfg == 4:
        return make_config4(seed, b_ids, B, poison_invalid)
    shp = dict(CONFIG_SHAPES[cfg])
    if R is not None: shp["R"] = R
    if A is not None: shp["A"] = A
    if T is not None: shp["T"] = T
    seed = MASTER_SEED + cfg if seed is None else seed
    b = np.arange(shp["B"] if B is None else B) if b_ids is None else np.asarray(b_ids, dtype=np.int64)
    log, rg = make_street_scenarios(seed, b, shp["A"], shp["R"], shp["T"], poison_invalid=poison_invalid)
    t0 = HISTORY - 1
    valid_t0 = log["valid"][:, t0, :]
    out = dict(config=cfg, seed=seed, b_ids=b, log=log, roadgraph=rg, t0=t0)
    if cfg == 2:
        act, av = delta_actions(seed, b, shp["A"], valid_t0)
        out.update(actions=act, action_valid=av, dynamics="delta_local", n_steps=1)
    elif cfg == 3:
        out.update(actions=None, action_valid=None, dynamics=None, n_steps=0)
    else:
        ns = 80 if n_steps is None else n_steps
        act, av = bicycle_actions(seed, b, shp["A"], ns, valid_t0)
        out.update(actions=act, action_valid=av, dynamics="bicycle", n_steps=ns)
    return out


def make_paths(log, extend=16, spacing=1.0):
    """One synthetic on-route path per agent (stand-in for the paper's roadgraph paths, L84): the
    agent's valid logged positions in time order, then `extend` more points straight ahead of the
    last logged heading at `spacing` metres.  arc_len = cumulative chord length from the first
    point (float64 sum, one rounding to float32).  Returns x, y, arc_len [B][A][P], valid [B][A][P],
    P = T + extend.  Input construction only: nothing here belongs to a metric."""
    B, T, A = log["x"].shape
    P = T + extend
    v = np.transpose(log["valid"], (0, 2, 1)) == 1                         # [B][A][T]
    x = np.transpose(log["x"], (0, 2, 1)).astype(np.float64); y = np.transpose(log["y"], (0, 2, 1)).astype(np.float64)
    yaw = np.transpose(log["yaw"], (0, 2, 1)).astype(np.float64)
    order = np.argsort(~v, axis=2, kind="stable")                          # valid rows first, in time order
    n = v.sum(axis=2)                                                      # [B][A] number of logged points
    gx = np.take_along_axis(x, order, 2); gy = np.take_along_axis(y, order, 2); gth = np.take_along_axis(yaw, order, 2)
    last = np.maximum(n - 1, 0)[..., None]
    lx = np.take_along_axis(gx, last, 2); ly = np.take_along_axis(gy, last, 2); lth = np.take_along_axis(gth, last, 2)
    j = np.arange(P)[None, None, :]
    e = np.maximum(j - (n[..., None] - 1), 0) * spacing                    # metres beyond the last logged point
    jj = np.minimum(j, T - 1)
    px = np.where(j < n[..., None], np.take_along_axis(gx, np.broadcast_to(jj, (B, A, P)), 2), lx + e * np.cos(lth))
    py = np.where(j < n[..., None], np.take_along_axis(gy, np.broadcast_to(jj, (B, A, P)), 2), ly + e * np.sin(lth))
    ok = (j < n[..., None] + extend) & (n[..., None] > 0)
    px = np.where(ok, px, 0.0); py = np.where(ok, py, 0.0)
    seg = np.hypot(np.diff(px, axis=2), np.diff(py, axis=2)) * ok[..., 1:]
    arc = np.concatenate([np.zeros((B, A, 1)), np.cumsum(seg, axis=2)], axis=2) * ok
    return dict(x=px.astype(np.float32), y=py.astype(np.float32), arc_len=arc.astype(np.float32), valid=ok.astype(np.uint8))
