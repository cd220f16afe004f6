"""Small helpers shared by the tests (array plumbing only; no method arithmetic)."""
import numpy as np

TRAJ_F = ("x", "y", "yaw", "vel_x", "vel_y", "length", "width")


def mk_traj(B, T, A, valid=0):
    tr = {k: np.zeros((B, T, A), np.float32) for k in TRAJ_F}
    tr["valid"] = np.full((B, T, A), valid, np.uint8)
    return tr


def set_agent(tr, b, t, a, x=0.0, y=0.0, yaw=0.0, vx=0.0, vy=0.0, length=4.5, width=2.0, valid=1):
    for k, v in zip(TRAJ_F, (x, y, yaw, vx, vy, length, width)):
        tr[k][b, t, a] = v
    tr["valid"][b, t, a] = valid


def boxes_traj(boxes):
    """boxes: list of (x, y, yaw, L, W) -> one scenario, T=1."""
    A = len(boxes)
    tr = mk_traj(1, 1, A, valid=1)
    for a, (x, y, yaw, L, W) in enumerate(boxes):
        set_agent(tr, 0, 0, a, x, y, yaw, 0, 0, L, W)
    return tr


def mk_roadgraph(polylines, B=1, R=None, types=None):
    """polylines: list of [n_i, 2] arrays (one scenario, replicated B times).
    dir_i = unit(p[i+1]-p[i]), last copies predecessor; id = polyline number."""
    xs, ys, dx, dy, ty, ids = [], [], [], [], [], []
    for pi, p in enumerate(polylines):
        p = np.asarray(p, np.float64)
        if len(p) > 1:
            d = p[1:] - p[:-1]
            n = np.linalg.norm(d, axis=1, keepdims=True)
            d = d / np.where(n > 0, n, 1)
            d = np.concatenate([d, d[-1:]], 0)
        else:
            d = np.array([[1.0, 0.0]])
        xs += list(p[:, 0]); ys += list(p[:, 1]); dx += list(d[:, 0]); dy += list(d[:, 1])
        ty += [2 if types is None else types[pi]] * len(p); ids += [pi] * len(p)
    n = len(xs)
    R = n if R is None else R
    rg = {"x": np.zeros((B, R), np.float32), "y": np.zeros((B, R), np.float32),
          "dir_x": np.ones((B, R), np.float32), "dir_y": np.zeros((B, R), np.float32),
          "type": np.zeros((B, R), np.int32), "id": np.full((B, R), -1, np.int32),
          "valid": np.zeros((B, R), np.uint8)}
    rg["x"][:, :n] = xs; rg["y"][:, :n] = ys; rg["dir_x"][:, :n] = dx; rg["dir_y"][:, :n] = dy
    rg["type"][:, :n] = ty; rg["id"][:, :n] = ids; rg["valid"][:, :n] = 1
    return rg


def rigid(tr, rg, phi, tx, ty):
    """Apply a common rigid transform to a trajectory dict and a roadgraph dict (float64 math)."""
    c, s = np.cos(phi), np.sin(phi)
    out = {k: v.copy() for k, v in tr.items()}
    x, y = tr["x"].astype(np.float64), tr["y"].astype(np.float64)
    out["x"] = (c * x - s * y + tx).astype(np.float32)
    out["y"] = (s * x + c * y + ty).astype(np.float32)
    out["yaw"] = (tr["yaw"].astype(np.float64) + phi).astype(np.float32)
    vx, vy = tr["vel_x"].astype(np.float64), tr["vel_y"].astype(np.float64)
    out["vel_x"] = (c * vx - s * vy).astype(np.float32)
    out["vel_y"] = (s * vx + c * vy).astype(np.float32)
    org = None
    if rg is not None:
        org = {k: v.copy() for k, v in rg.items()}
        x, y = rg["x"].astype(np.float64), rg["y"].astype(np.float64)
        org["x"] = (c * x - s * y + tx).astype(np.float32)
        org["y"] = (s * x + c * y + ty).astype(np.float32)
        dx, dy = rg["dir_x"].astype(np.float64), rg["dir_y"].astype(np.float64)
        org["dir_x"] = (c * dx - s * dy).astype(np.float32)
        org["dir_y"] = (s * dx + c * dy).astype(np.float32)
    return out, org
