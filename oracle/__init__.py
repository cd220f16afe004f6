"""ORACLE — TEST INFRASTRUCTURE ONLY (see wm_oracle.cpp header).

ctypes binding of the scalar C++ CPU oracle.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package; the product
package never does.  Inputs/outputs are numpy arrays in the layouts of the paper's state
definition as fixed by the C-ABI (time-major [B][T][A], roadgraph [B][R]).
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "wm_oracle.cpp")
_LIB = os.path.join(_HERE, "libwm_oracle.so")

DYN_BICYCLE = 0
DYN_DELTA_LOCAL = 1
DYN_DELTA_GLOBAL = 2
BAND = 1e-4  # ambiguity band in metres (BASELINE.json north_star)

TRAJ_F = ("x", "y", "yaw", "vel_x", "vel_y", "length", "width")
RG_F = ("x", "y", "dir_x", "dir_y")


def build(force=False):
    """Compile wm_oracle.cpp -> libwm_oracle.so (g++ -O2, OpenMP over scenarios)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    cmd = ["g++", "-O2", "-fopenmp", "-ffp-contract=off", "-std=c++17", "-shared", "-fPIC",
           "-o", _LIB, _SRC]
    subprocess.check_call(cmd)
    return _LIB


class _Traj(C.Structure):
    _fields_ = [("B", C.c_int32), ("A", C.c_int32), ("T", C.c_int32)] + \
               [(k, C.c_void_p) for k in TRAJ_F] + [("valid", C.c_void_p)]


class _Rg(C.Structure):
    _fields_ = [("B", C.c_int32), ("R", C.c_int32)] + [(k, C.c_void_p) for k in RG_F] + \
               [("type", C.c_void_p), ("id", C.c_void_p), ("valid", C.c_void_p)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        # WM_ORACLE_LIB: another build of the SAME source (tests/test_sanitizers.py loads an ASan / UBSan build)
        _lib = C.CDLL(os.environ.get("WM_ORACLE_LIB") or build())
        _lib.orc_count_segments.restype = C.c_int32
        _lib.orc_num_threads.restype = C.c_int32
    return _lib


def num_threads():
    return int(lib().orc_num_threads())


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _check(a, dtype, shape):
    assert a.dtype == dtype and a.flags["C_CONTIGUOUS"] and tuple(a.shape) == tuple(shape), \
        (a.dtype, a.shape, dtype, shape)


def _traj(tr):
    B, T, A = tr["x"].shape
    for k in TRAJ_F:
        _check(tr[k], np.float32, (B, T, A))
    _check(tr["valid"], np.uint8, (B, T, A))
    s = _Traj(B, A, T, *[_p(tr[k]) for k in TRAJ_F], _p(tr["valid"]))
    return s, (B, T, A)


def _rg(rg):
    B, R = rg["x"].shape
    for k in RG_F:
        _check(rg[k], np.float32, (B, R))
    _check(rg["type"], np.int32, (B, R)); _check(rg["id"], np.int32, (B, R))
    _check(rg["valid"], np.uint8, (B, R))
    return _Rg(B, R, *[_p(rg[k]) for k in RG_F], _p(rg["type"]), _p(rg["id"]), _p(rg["valid"])), (B, R)


def copy_traj(tr):
    return {k: np.ascontiguousarray(v).copy() for k, v in tr.items()}


def empty_like_traj(tr):
    return {k: np.zeros_like(v) for k, v in tr.items()}


def reset(log, history=11):
    sim = empty_like_traj(log)
    ls, _ = _traj(log); ss, _ = _traj(sim)
    lib().orc_reset(C.byref(ls), C.byref(ss), C.c_int32(history))
    return sim


def step(log, sim, t, dynamics, action, action_valid, dt=0.1, max_accel=6.0, max_curvature=0.3):
    """In place: writes sim row t+1. action [B][C][A] float32, action_valid [B][A] uint8."""
    ls, (B, T, A) = _traj(log); ss, _ = _traj(sim)
    Cn = 2 if dynamics == DYN_BICYCLE else 3
    _check(action, np.float32, (B, Cn, A)); _check(action_valid, np.uint8, (B, A))
    lib().orc_step(C.byref(ls), C.byref(ss), C.c_int32(t), C.c_int32(dynamics), C.c_double(dt),
                   C.c_double(max_accel), C.c_double(max_curvature), _p(action), C.c_int64(Cn * A),
                   _p(action_valid), C.c_int64(A))
    return sim


def overlap(sim, t, want_gap=True, want_pair=True):
    ss, (B, T, A) = _traj(sim)
    gap = np.empty((B, A, A), np.float64) if want_gap else None
    pair = np.empty((B, A, A), np.uint8) if want_pair else None
    flag = np.empty((B, A), np.uint8)
    lib().orc_overlap(C.byref(ss), C.c_int32(t), _p(gap), _p(pair), _p(flag))
    return dict(gap=gap, pair=pair, flag=flag)


def offroad(sim, t, rg, band=BAND, details=True):
    ss, (B, T, A) = _traj(sim); rs, _ = _rg(rg)
    sd = np.empty((B, A), np.float32); flag = np.empty((B, A), np.uint8)
    csd = np.empty((B, 4, A), np.float32) if details else None
    amb = np.empty((B, 4, A), np.uint8) if details else None
    win = np.empty((B, 4, A), np.int32) if details else None
    lib().orc_offroad(C.byref(ss), C.c_int32(t), C.byref(rs), C.c_double(band), _p(sd), _p(csd),
                      _p(flag), _p(amb), _p(win))
    return dict(signed_dist=sd, corner_dist=csd, flag=flag, ambig=amb, win_seg=win)


def count_segments(rg, b):
    rs, _ = _rg(rg)
    return int(lib().orc_count_segments(C.byref(rs), C.c_int32(b)))


def log_divergence(log, sim, t):
    ls, (B, T, A) = _traj(log); ss, _ = _traj(sim)
    d = np.empty((B, A), np.float32); v = np.empty((B, A), np.uint8)
    lib().orc_log_divergence(C.byref(ls), C.byref(ss), C.c_int32(t), _p(d), _p(v))
    return dict(dist=d, valid=v)


def observe_history(sim, t, H=11):
    ss, (B, T, A) = _traj(sim)
    hist = np.empty((B, A, H, 7, A), np.float32); hv = np.empty((B, A, H, A), np.uint8)
    lib().orc_observe_history(C.byref(ss), C.c_int32(t), C.c_int32(H), _p(hist), _p(hv))
    return dict(hist=hist, hist_valid=hv)


def observe_topk(sim, rg, t, k, order=0):
    """order 0: ascending roadgraph index (D24); 1: ascending (distance key, index) (D44)."""
    ss, (B, T, A) = _traj(sim); rs, _ = _rg(rg)
    idx = np.empty((B, A, k), np.int32); feat = np.empty((B, A, 4, k), np.float32)
    typ = np.empty((B, A, k), np.int32); kth = np.empty((B, A), np.float32)
    lib().orc_observe_topk(C.byref(ss), C.byref(rs), C.c_int32(t), C.c_int32(k), C.c_int32(order), _p(idx), _p(feat),
                           _p(typ), _p(kth))
    return dict(rg_index=idx, rg_feat=feat, rg_type=typ, kth_key=kth)


def rollout(log, sim, rg, t0, n_steps, dynamics, actions, action_valid, dt=0.1, max_accel=6.0,
            max_curvature=0.3, band=BAND):
    """In place on sim rows t0+1..t0+n_steps. actions [B][n_steps][C][A]."""
    ls, (B, T, A) = _traj(log); ss, _ = _traj(sim); rs, _ = _rg(rg)
    Cn = 2 if dynamics == DYN_BICYCLE else 3
    _check(actions, np.float32, (B, n_steps, Cn, A)); _check(action_valid, np.uint8, (B, n_steps, A))
    out = dict(overlap=np.empty((B, n_steps, A), np.uint8), offroad=np.empty((B, n_steps, A), np.uint8),
               offroad_dist=np.empty((B, n_steps, A), np.float32), log_div=np.empty((B, n_steps, A), np.float32),
               any_overlap=np.empty((B, A), np.uint8), any_offroad=np.empty((B, A), np.uint8),
               ade=np.empty((B, A), np.float32))
    lib().orc_rollout(C.byref(ls), C.byref(ss), C.byref(rs), C.c_int32(t0), C.c_int32(n_steps),
                      C.c_int32(dynamics), C.c_double(dt), C.c_double(max_accel), C.c_double(max_curvature),
                      _p(actions), _p(action_valid), C.c_double(band), _p(out["overlap"]), _p(out["offroad"]),
                      _p(out["offroad_dist"]), _p(out["log_div"]), _p(out["any_overlap"]),
                      _p(out["any_offroad"]), _p(out["ade"]))
    return out


def expert_actions(tr, t, n_steps, dynamics, dt=0.1):
    """O9: inverse kinematics on rows t+s, t+s+1 (L335 / Eq. 3). action [B][n_steps][C][A]."""
    ts, (B, T, A) = _traj(tr)
    Cn = 2 if dynamics == DYN_BICYCLE else 3
    act = np.empty((B, n_steps, Cn, A), np.float32); val = np.empty((B, n_steps, A), np.uint8)
    den = np.empty((B, n_steps, A), np.float64)
    lib().orc_expert_actions(C.byref(ts), C.c_int32(t), C.c_int32(n_steps), C.c_int32(dynamics), C.c_double(dt),
                             _p(act), _p(val), _p(den))
    return dict(action=act, valid=val, kden=den)


def kinematic(tr, t, n_steps=1, dt=0.1, max_accel=6.0, max_curvature=0.3):
    """O10: kinematic infeasibility of the transitions into rows t..t+n_steps-1 (L104)."""
    ts, (B, T, A) = _traj(tr)
    shp = (B, n_steps, A)
    acc = np.empty(shp, np.float32); cur = np.empty(shp, np.float32); den = np.empty(shp, np.float64)
    flag = np.empty(shp, np.uint8); val = np.empty(shp, np.uint8)
    lib().orc_kinematic(C.byref(ts), C.c_int32(t), C.c_int32(n_steps), C.c_double(dt), C.c_double(max_accel),
                        C.c_double(max_curvature), _p(acc), _p(cur), _p(den), _p(flag), _p(val))
    return dict(accel=acc, curvature=cur, kden=den, flag=flag, valid=val)


class _Paths(C.Structure):
    _fields_ = [("B", C.c_int32), ("A", C.c_int32), ("P", C.c_int32), ("x", C.c_void_p), ("y", C.c_void_p),
                ("arc_len", C.c_void_p), ("valid", C.c_void_p)]


def route_progress(log, sim, t, paths):
    """O11 (L96). paths: dict x, y, arc_len float32 [B][A][P], valid uint8 [B][A][P]."""
    ls, (B, T, A) = _traj(log); ss, _ = _traj(sim)
    P = paths["x"].shape[2]
    for k in ("x", "y", "arc_len"):
        _check(paths[k], np.float32, (B, A, P))
    _check(paths["valid"], np.uint8, (B, A, P))
    ps = _Paths(B, A, P, _p(paths["x"]), _p(paths["y"]), _p(paths["arc_len"]), _p(paths["valid"]))
    ratio = np.empty((B, A), np.float32); val = np.empty((B, A), np.uint8); cl = np.empty((B, 3, A), np.int32)
    lib().orc_route_progress(C.byref(ls), C.byref(ss), C.c_int32(t), C.byref(ps), _p(ratio), _p(val), _p(cl))
    return dict(ratio=ratio, valid=val, closest=cl)


def _paths(paths, B, A):
    P = paths["x"].shape[2]
    for k in ("x", "y", "arc_len"):
        _check(paths[k], np.float32, (B, A, P))
    _check(paths["valid"], np.uint8, (B, A, P))
    return _Paths(B, A, P, _p(paths["x"]), _p(paths["y"]), _p(paths["arc_len"]), _p(paths["valid"]))


def offroute(sim, t, on_route, off_route, max_dist, margin):
    """O12 (L98; thresholds are arguments, D36). off_route may be None."""
    ss, (B, T, A) = _traj(sim)
    on = _paths(on_route, B, A)
    off = _paths(off_route, B, A) if off_route is not None else None
    d = np.empty((B, A), np.float32); f = np.empty((B, A), np.uint8)
    lib().orc_offroute(C.byref(ss), C.c_int32(t), C.byref(on), C.byref(off) if off is not None else None,
                       C.c_float(max_dist), C.c_float(margin), _p(d), _p(f))
    return dict(dist_on=d, flag=f)


class _Idm(C.Structure):
    _fields_ = [(k, C.c_float) for k in ("v0", "T", "s0", "a_max", "b", "delta", "b_max")]


IDM_DEFAULTS = dict(v0=30.0, T=1.5, s0=2.0, a_max=1.0, b=1.5, delta=4.0, b_max=4.0)   # D37: declared, not from the paper


def idm_step(sim, t, paths, idm_valid, dt=0.1, **params):
    """O13: in place, writes row t+1 of the IDM-controlled agents (L110-L112; readings D37-D41)."""
    ss, (B, T, A) = _traj(sim)
    pa = _paths(paths, B, A)
    _check(idm_valid, np.uint8, (B, A))
    prm = dict(IDM_DEFAULTS); prm.update(params)
    ps = _Idm(*[prm[k] for k in ("v0", "T", "s0", "a_max", "b", "delta", "b_max")])
    acc = np.empty((B, A), np.float32); lead = np.empty((B, A), np.int32)
    lib().orc_idm_step(C.byref(ss), C.c_int32(t), C.byref(pa), _p(idm_valid), C.byref(ps), C.c_double(dt), _p(acc), _p(lead))
    return dict(accel=acc, lead=lead)


def rollout_vjp(sim, t0, n_steps, dynamics, actions, action_valid, g_rows, dt=0.1, max_accel=6.0, max_curvature=0.3):
    """O14: reverse-mode derivative of the rollout's dynamics (L252).  g_rows [B][n_steps][5][A] float32 = cotangents
    of rows t0+1..t0+n_steps (x, y, yaw, vel_x, vel_y).  Returns g_actions [B][n_steps][C][A], g_state0 [B][5][A]."""
    ss, (B, T, A) = _traj(sim)
    Cn = 2 if dynamics == DYN_BICYCLE else 3
    _check(actions, np.float32, (B, n_steps, Cn, A)); _check(action_valid, np.uint8, (B, n_steps, A))
    _check(g_rows, np.float32, (B, n_steps, 5, A))
    ga = np.empty((B, n_steps, Cn, A), np.float32); g0 = np.empty((B, 5, A), np.float32)
    lib().orc_rollout_vjp(C.byref(ss), C.c_int32(t0), C.c_int32(n_steps), C.c_int32(dynamics), C.c_double(dt), C.c_double(max_accel),
                          C.c_double(max_curvature), _p(actions), _p(action_valid), _p(g_rows), _p(ga), _p(g0))
    return dict(g_actions=ga, g_state0=g0)


class _Grid(C.Structure):
    _fields_ = [("n", C.c_int32 * 3), ("lo", C.c_float * 3), ("hi", C.c_float * 3)]


def _grid(n, lo, hi):
    g = _Grid()
    for c in range(3):
        g.n[c] = int(n[c]) if c < len(n) else 1
        g.lo[c] = float(lo[c]) if c < len(lo) else 0.0
        g.hi[c] = float(hi[c]) if c < len(hi) else 0.0
    return g


def discretize_actions(action, n, lo, hi, valid=None):
    """O15 (L204, D42): action [..., C, A] float32 -> joint bin index [..., A] int32 and the de-quantised action."""
    Cn, A = action.shape[-2:]
    N = int(np.prod(action.shape[:-2], dtype=np.int64))
    act = np.ascontiguousarray(action, np.float32)
    idx = np.empty(action.shape[:-2] + (A,), np.int32); deq = np.empty_like(act)
    v = None if valid is None else np.ascontiguousarray(valid, np.uint8)
    g = _grid(n, lo, hi)
    lib().orc_discretize_actions(C.byref(g), C.c_int32(Cn), C.c_int64(N), C.c_int32(A), _p(act), _p(v), _p(idx), _p(deq))
    return dict(index=idx, action=deq)


def actions_from_index(index, Cn, n, lo, hi):
    A = index.shape[-1]
    N = int(np.prod(index.shape[:-1], dtype=np.int64))
    idx = np.ascontiguousarray(index, np.int32)
    act = np.empty(index.shape[:-1] + (Cn, A), np.float32)
    g = _grid(n, lo, hi)
    lib().orc_actions_from_index(C.byref(g), C.c_int32(Cn), C.c_int64(N), C.c_int32(A), _p(idx), _p(act))
    return act
