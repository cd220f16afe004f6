"""Thin Python binding of the C-ABI in include/wm.h (same names, argument marshalling only).

Every step of the path runs in the CUDA kernels of libwm_b200.so; PyTorch is used to own
device memory and streams.  There is no CPU or eager fallback: if the shared library is
missing or a call fails, this module raises.
"""
import ctypes as C
import os

import torch

from . import _build

WM_OK, WM_ERR_ARG, WM_ERR_CUDA, WM_ERR_UNSUPPORTED, WM_ERR_STATE, WM_ERR_TOO_LARGE = 0, -1, -2, -3, -4, -5
WM_STATIC_MAX_B, WM_STATIC_MAX_POINTS = 64, 1 << 20
WM_DYN_INVERTIBLE_BICYCLE, WM_DYN_DELTA_LOCAL, WM_DYN_DELTA_GLOBAL = 0, 1, 2
WM_TYPE_LANE, WM_TYPE_ROAD_EDGE = 1, 2
WM_OFFROAD_CULLED, WM_OFFROAD_BRUTE_FORCE = 0, 1
WM_ROLLOUT_FUSED, WM_ROLLOUT_STEPWISE = 0, 1
WM_TOPK_BY_INDEX, WM_TOPK_BY_DISTANCE = 0, 1
_ERR = {-1: "WM_ERR_ARG", -2: "WM_ERR_CUDA", -3: "WM_ERR_UNSUPPORTED", -4: "WM_ERR_STATE", -5: "WM_ERR_TOO_LARGE"}

TRAJ_F = ("x", "y", "yaw", "vel_x", "vel_y", "length", "width")
RG_F = ("x", "y", "dir_x", "dir_y")

EXPORTS = ("wm_create", "wm_destroy", "wm_last_cuda_error", "wm_version", "wm_prepare", "wm_reset",
           "wm_step", "wm_metrics_overlap", "wm_metrics_offroad", "wm_log_divergence", "wm_observe",
           "wm_expert_actions", "wm_metrics_kinematic", "wm_metrics_route_progress", "wm_metrics_offroute", "wm_idm_step", "wm_rollout", "wm_rollout_host", "wm_segment_counts", "wm_kernel_launches", "wm_offroad_stats", "wm_offroad_stats_enable", "wm_grid_stats",
           "wm_discretize_actions", "wm_actions_from_index", "wm_expert_actions_discrete", "wm_rollout_vjp", "wm_step_vjp", "wm_rollout_kernel_times", "wm_selftest_ffma", "wm_observe_topk_static")


class wm_traj(C.Structure):
    _fields_ = [("B", C.c_int32), ("A", C.c_int32), ("T", C.c_int32)] + \
               [(k, C.c_void_p) for k in TRAJ_F] + [("valid", C.c_void_p)]


class wm_roadgraph(C.Structure):
    _fields_ = [("B", C.c_int32), ("R", C.c_int32)] + [(k, C.c_void_p) for k in RG_F] + \
               [("type", C.c_void_p), ("id", C.c_void_p), ("valid", C.c_void_p)]


class wm_config(C.Structure):
    _fields_ = [("dynamics", C.c_int32), ("dt", C.c_float), ("max_accel", C.c_float),
                ("max_curvature", C.c_float), ("history", C.c_int32), ("topk", C.c_int32),
                ("offroad_mode", C.c_int32), ("rollout_mode", C.c_int32), ("topk_order", C.c_int32)]


class wm_rollout_out(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("overlap", "offroad", "offroad_dist", "log_div",
                                           "any_overlap", "any_offroad", "ade")]


_lib = None


def lib_path():
    return _build.LIB


def load():
    """dlopen libwm_b200.so (building it first if the sources are newer). Raises if absent."""
    global _lib
    if _lib is None:
        # WM_B200_LIB: another build of the SAME sources (the host-sanitizer test loads libwm_b200_san.so)
        path = os.environ.get("WM_B200_LIB") or _build.build()
        if not os.path.exists(path):
            raise RuntimeError("libwm_b200.so is missing: the CUDA extension must be built (no fallback)")
        _lib = C.CDLL(path)
        _lib.wm_version.restype = C.c_char_p
        _lib.wm_kernel_launches.restype = C.c_int64
        _lib.wm_kernel_launches.argtypes = [C.c_void_p]
        for name in EXPORTS:
            getattr(_lib, name)
    return _lib


class WmError(RuntimeError):
    pass


def _check(rc, what):
    if rc != WM_OK:
        extra = ""
        if rc == WM_ERR_CUDA:
            extra = " (cudaError_t %d)" % load().wm_last_cuda_error()
        raise WmError("%s failed: %s%s" % (what, _ERR.get(rc, rc), extra))


def _ptr(t, dtype=None, device_type="cuda"):
    if t is None:
        return None
    assert isinstance(t, torch.Tensor) and t.is_contiguous(), "contiguous torch tensor expected"
    assert t.device.type == device_type, "tensor on %s expected, got %s" % (device_type, t.device)
    if dtype is not None:
        assert t.dtype == dtype, (t.dtype, dtype)
    return C.c_void_p(t.data_ptr())


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def traj_struct(tr, device_type="cuda"):
    """dict of [B][T][A] tensors -> wm_traj."""
    B, T, A = tr["x"].shape
    for k in TRAJ_F:
        assert tuple(tr[k].shape) == (B, T, A)
    return wm_traj(B, A, T, *[_ptr(tr[k], torch.float32, device_type) for k in TRAJ_F],
                   _ptr(tr["valid"], torch.uint8, device_type))


def roadgraph_struct(rg, device_type="cuda"):
    B, R = rg["x"].shape
    return wm_roadgraph(B, R, *[_ptr(rg[k], torch.float32, device_type) for k in RG_F],
                        _ptr(rg["type"], torch.int32, device_type), _ptr(rg["id"], torch.int32, device_type),
                        _ptr(rg["valid"], torch.uint8, device_type))


def rollout_out_struct(out, device_type="cuda"):
    dt = dict(overlap=torch.uint8, offroad=torch.uint8, offroad_dist=torch.float32, log_div=torch.float32,
              any_overlap=torch.uint8, any_offroad=torch.uint8, ade=torch.float32)
    return wm_rollout_out(*[_ptr(out.get(k), dt[k], device_type) for k in dt])


# ---- the entry points, same names as the C-ABI ----
def wm_version():
    return load().wm_version().decode()


def wm_create(dynamics=WM_DYN_INVERTIBLE_BICYCLE, dt=0.1, max_accel=6.0, max_curvature=0.3, history=11, topk=1000,
              offroad_mode=WM_OFFROAD_CULLED, rollout_mode=WM_ROLLOUT_FUSED, topk_order=WM_TOPK_BY_INDEX):
    h = C.c_void_p()
    cfg = wm_config(dynamics, dt, max_accel, max_curvature, history, topk, offroad_mode, rollout_mode, topk_order)
    _check(load().wm_create(C.byref(h), C.byref(cfg)), "wm_create")
    return h


def wm_destroy(h):
    _check(load().wm_destroy(h), "wm_destroy")


def wm_prepare(h, rg, stream=None):
    n = C.c_int32(0)
    s = roadgraph_struct(rg)
    _check(load().wm_prepare(h, C.byref(s), C.byref(n), _stream(stream)), "wm_prepare")
    return n.value


def wm_reset(h, log, sim, stream=None):
    t = C.c_int32(0)
    ls, ss = traj_struct(log), traj_struct(sim)
    _check(load().wm_reset(h, C.byref(ls), C.byref(ss), C.byref(t), _stream(stream)), "wm_reset")
    return t.value


def wm_step(h, log, sim, t, action, action_valid, stream=None):
    ls, ss = traj_struct(log), traj_struct(sim)
    _check(load().wm_step(h, C.byref(ls), C.byref(ss), C.c_int32(t), _ptr(action, torch.float32),
                          _ptr(action_valid, torch.uint8), _stream(stream)), "wm_step")


def wm_metrics_overlap(h, sim, t, pair_bits, agent_flag, stream=None):
    ss = traj_struct(sim)
    _check(load().wm_metrics_overlap(h, C.byref(ss), C.c_int32(t), _ptr(pair_bits, torch.int32),
                                     _ptr(agent_flag, torch.uint8), _stream(stream)), "wm_metrics_overlap")


def wm_metrics_offroad(h, sim, t, signed_dist, corner_dist, agent_flag, stream=None):
    ss = traj_struct(sim)
    _check(load().wm_metrics_offroad(h, C.byref(ss), C.c_int32(t), _ptr(signed_dist, torch.float32),
                                     _ptr(corner_dist, torch.float32), _ptr(agent_flag, torch.uint8),
                                     _stream(stream)), "wm_metrics_offroad")


def wm_log_divergence(h, log, sim, t, dist, valid, stream=None):
    ls, ss = traj_struct(log), traj_struct(sim)
    _check(load().wm_log_divergence(h, C.byref(ls), C.byref(ss), C.c_int32(t), _ptr(dist, torch.float32),
                                    _ptr(valid, torch.uint8), _stream(stream)), "wm_log_divergence")


def wm_expert_actions(h, tr, t, n_steps, action, action_valid, stream=None):
    ts = traj_struct(tr)
    _check(load().wm_expert_actions(h, C.byref(ts), C.c_int32(t), C.c_int32(n_steps), _ptr(action, torch.float32),
                                    _ptr(action_valid, torch.uint8), _stream(stream)), "wm_expert_actions")


def wm_metrics_kinematic(h, sim, t, n_steps, accel, curvature, flag, stream=None):
    ss = traj_struct(sim)
    _check(load().wm_metrics_kinematic(h, C.byref(ss), C.c_int32(t), C.c_int32(n_steps), _ptr(accel, torch.float32),
                                       _ptr(curvature, torch.float32), _ptr(flag, torch.uint8), _stream(stream)), "wm_metrics_kinematic")


class wm_paths(C.Structure):
    _fields_ = [("B", C.c_int32), ("A", C.c_int32), ("P", C.c_int32), ("x", C.c_void_p), ("y", C.c_void_p),
                ("arc_len", C.c_void_p), ("valid", C.c_void_p)]


class wm_action_grid(C.Structure):
    _fields_ = [("n", C.c_int32 * 3), ("lo", C.c_float * 3), ("hi", C.c_float * 3)]


def action_grid(n, lo, hi):
    g = wm_action_grid()
    for c in range(3):
        g.n[c] = int(n[c]) if c < len(n) else 1
        g.lo[c] = float(lo[c]) if c < len(lo) else 0.0
        g.hi[c] = float(hi[c]) if c < len(hi) else 0.0
    return g


def wm_discretize_actions(h, grid, action, index, dequant=None, valid=None, stream=None):
    """action [..., C, A] -> index [..., A] int32, dequant like action (may be the same tensor)."""
    A = action.shape[-1]
    N = index.numel() // A
    _check(load().wm_discretize_actions(h, C.byref(grid), C.c_int64(N), C.c_int32(A), _ptr(action, torch.float32),
                                        _ptr(valid, torch.uint8), _ptr(index, torch.int32), _ptr(dequant, torch.float32),
                                        _stream(stream)), "wm_discretize_actions")


def wm_actions_from_index(h, grid, index, action, stream=None):
    A = index.shape[-1]
    N = index.numel() // A
    _check(load().wm_actions_from_index(h, C.byref(grid), C.c_int64(N), C.c_int32(A), _ptr(index, torch.int32),
                                        _ptr(action, torch.float32), _stream(stream)), "wm_actions_from_index")


def wm_expert_actions_discrete(h, tr, t, n_steps, grid, index, action, action_valid, stream=None):
    ts = traj_struct(tr)
    _check(load().wm_expert_actions_discrete(h, C.byref(ts), C.c_int32(t), C.c_int32(n_steps), C.byref(grid), _ptr(index, torch.int32),
                                             _ptr(action, torch.float32), _ptr(action_valid, torch.uint8), _stream(stream)),
           "wm_expert_actions_discrete")


def wm_rollout_vjp(h, sim, t0, n_steps, actions, action_valid, g_rows, g_actions, g_state0=None, stream=None):
    ss = traj_struct(sim)
    _check(load().wm_rollout_vjp(h, C.byref(ss), C.c_int32(t0), C.c_int32(n_steps), _ptr(actions, torch.float32),
                                 _ptr(action_valid, torch.uint8), _ptr(g_rows, torch.float32), _ptr(g_actions, torch.float32),
                                 _ptr(g_state0, torch.float32), _stream(stream)), "wm_rollout_vjp")


def wm_step_vjp(h, sim, t, action, action_valid, g_next, g_state, g_action, stream=None):
    ss = traj_struct(sim)
    _check(load().wm_step_vjp(h, C.byref(ss), C.c_int32(t), _ptr(action, torch.float32), _ptr(action_valid, torch.uint8),
                              _ptr(g_next, torch.float32), _ptr(g_state, torch.float32), _ptr(g_action, torch.float32),
                              _stream(stream)), "wm_step_vjp")


def paths_struct(paths):
    """paths: dict of device tensors x, y, arc_len float32 [B][A][P], valid uint8 [B][A][P]."""
    B, A, P = paths["x"].shape
    return wm_paths(B, A, P, _ptr(paths["x"], torch.float32), _ptr(paths["y"], torch.float32), _ptr(paths["arc_len"], torch.float32),
                    _ptr(paths["valid"], torch.uint8))


def wm_metrics_offroute(h, sim, t, on_route, off_route, max_dist, margin, dist_on, flag, stream=None):
    ss, on = traj_struct(sim), paths_struct(on_route)
    off = paths_struct(off_route) if off_route is not None else None
    _check(load().wm_metrics_offroute(h, C.byref(ss), C.c_int32(t), C.byref(on), C.byref(off) if off is not None else None,
                                      C.c_float(max_dist), C.c_float(margin), _ptr(dist_on, torch.float32), _ptr(flag, torch.uint8),
                                      _stream(stream)), "wm_metrics_offroute")


class wm_idm_params(C.Structure):
    _fields_ = [(k, C.c_float) for k in ("v0", "T", "s0", "a_max", "b", "delta", "b_max")]


IDM_DEFAULTS = dict(v0=30.0, T=1.5, s0=2.0, a_max=1.0, b=1.5, delta=4.0, b_max=4.0)   # D37: declared, not from the paper


def wm_idm_step(h, sim, t, paths, idm_valid, accel=None, lead=None, stream=None, **params):
    ss, ps = traj_struct(sim), paths_struct(paths)
    prm = dict(IDM_DEFAULTS); prm.update(params)
    q = wm_idm_params(*[prm[k] for k in ("v0", "T", "s0", "a_max", "b", "delta", "b_max")])
    _check(load().wm_idm_step(h, C.byref(ss), C.c_int32(t), C.byref(ps), _ptr(idm_valid, torch.uint8), C.byref(q),
                              _ptr(accel, torch.float32), _ptr(lead, torch.int32), _stream(stream)), "wm_idm_step")


def wm_metrics_route_progress(h, log, sim, t, paths, ratio, valid, stream=None):
    ls, ss = traj_struct(log), traj_struct(sim)
    ps = paths_struct(paths)
    _check(load().wm_metrics_route_progress(h, C.byref(ls), C.byref(ss), C.c_int32(t), C.byref(ps), _ptr(ratio, torch.float32),
                                            _ptr(valid, torch.uint8), _stream(stream)), "wm_metrics_route_progress")


def wm_observe(h, sim, rg, t, hist=None, hist_valid=None, rg_index=None, rg_feat=None, rg_type=None, stream=None):
    ss = traj_struct(sim)
    rs = roadgraph_struct(rg) if rg is not None else None
    _check(load().wm_observe(h, C.byref(ss), C.byref(rs) if rs is not None else None, C.c_int32(t),
                             _ptr(hist, torch.float32), _ptr(hist_valid, torch.uint8), _ptr(rg_index, torch.int32),
                             _ptr(rg_feat, torch.float32), _ptr(rg_type, torch.int32), _stream(stream)), "wm_observe")


def wm_observe_topk_static(sim, rg, t, topk, rg_index, rg_feat, rg_type, topk_order=WM_TOPK_BY_INDEX, stream=None):
    """Top-k observation without a handle and without any device allocation (see include/wm.h): for callers
    whose GPU memory is already spoken for (a framework's pooled allocator, a fixed start-up budget) or who
    cannot afford cudaMalloc's device-wide stall.  B <= WM_STATIC_MAX_B and B * R <= WM_STATIC_MAX_POINTS,
    else WmError(WM_ERR_TOO_LARGE).  All calls share one built-in scratch array per GPU: keep them on one stream."""
    ss, rs = traj_struct(sim), roadgraph_struct(rg)
    _check(load().wm_observe_topk_static(C.byref(ss), C.byref(rs), C.c_int32(t), C.c_int32(topk), C.c_int32(topk_order),
                                         _ptr(rg_index, torch.int32), _ptr(rg_feat, torch.float32),
                                         _ptr(rg_type, torch.int32), _stream(stream)), "wm_observe_topk_static")


def wm_rollout(h, log, sim, t0, n_steps, actions, action_valid, out, stream=None):
    ls, ss = traj_struct(log), traj_struct(sim)
    os_ = rollout_out_struct(out)
    _check(load().wm_rollout(h, C.byref(ls), C.byref(ss), C.c_int32(t0), C.c_int32(n_steps),
                             _ptr(actions, torch.float32), _ptr(action_valid, torch.uint8), C.byref(os_),
                             _stream(stream)), "wm_rollout")


def wm_rollout_kernel_times(h, log, sim, t0, n_steps, actions, action_valid, out, stream=None):
    """(ms of k_rollout_dyn, ms of k_rollout_metrics) of one eager run of the fused rollout."""
    ls, ss, os_ = traj_struct(log), traj_struct(sim), rollout_out_struct(out)
    ms = (C.c_float * 2)()
    _check(load().wm_rollout_kernel_times(h, C.byref(ls), C.byref(ss), C.c_int32(t0), C.c_int32(n_steps), _ptr(actions, torch.float32),
                                          _ptr(action_valid, torch.uint8), C.byref(os_), ms, _stream(stream)), "wm_rollout_kernel_times")
    return float(ms[0]), float(ms[1])


def wm_selftest_ffma(h, packed, ctas, iters, stream=None):
    """(ms, flop) of a register-resident FFMA / FFMA2 loop: the FP32 peak as measured on this GPU."""
    ms = C.c_float(0); fl = C.c_double(0)
    _check(load().wm_selftest_ffma(h, C.c_int32(int(packed)), C.c_int32(ctas), C.c_int32(iters), C.byref(ms), C.byref(fl), _stream(stream)),
           "wm_selftest_ffma")
    return float(ms.value), float(fl.value)


def wm_rollout_host(h, log_host, rg_host, n_steps, actions_host, action_valid_host, out_host, sim_host=None, stream=None):
    ls, rs = traj_struct(log_host, "cpu"), roadgraph_struct(rg_host, "cpu")
    os_ = rollout_out_struct(out_host, "cpu")
    sh = traj_struct(sim_host, "cpu") if sim_host is not None else None
    _check(load().wm_rollout_host(h, C.byref(ls), C.byref(rs), C.c_int32(n_steps),
                                  _ptr(actions_host, torch.float32, "cpu"), _ptr(action_valid_host, torch.uint8, "cpu"),
                                  C.byref(os_), C.byref(sh) if sh is not None else None, _stream(stream)),
           "wm_rollout_host")


def wm_segment_counts(h, B, stream=None):
    buf = (C.c_int32 * B)()
    _check(load().wm_segment_counts(h, buf, C.c_int32(B), _stream(stream)), "wm_segment_counts")
    return list(buf)


def wm_kernel_launches(h):
    return int(load().wm_kernel_launches(h))


def wm_offroad_stats(h, stream=None):
    """(pairs evaluated, brute-force pairs, slow-path corners, corners) of the exact grid search
    since the last call; counted only after wm_offroad_stats_enable(h, True)."""
    buf = (C.c_int64 * 4)()
    _check(load().wm_offroad_stats(h, buf, _stream(stream)), "wm_offroad_stats")
    return tuple(int(v) for v in buf)


def wm_grid_stats(h, stream=None):
    """Cells of the prepared search grids and how many have no candidate list (their queries search all segments):
    dict level -> (cells, cells without a list, share), levels inner / mid / outer, summed over the prepared scenarios."""
    buf = (C.c_int64 * 6)()
    _check(load().wm_grid_stats(h, buf, _stream(stream)), "wm_grid_stats")
    v = [int(x) for x in buf]
    return {k: (v[2 * i], v[2 * i + 1], v[2 * i + 1] / max(v[2 * i], 1)) for i, k in enumerate(("inner", "mid", "outer"))}


def wm_offroad_stats_enable(h, on=True):
    _check(load().wm_offroad_stats_enable(h, C.c_int32(1 if on else 0)), "wm_offroad_stats_enable")


# ---- small conveniences for tests / bench: torch allocation of the ABI's arrays ----
def to_device(d, device="cuda"):
    """numpy dict (wm_scenarios layout) -> dict of contiguous torch tensors on `device`."""
    return {k: torch.from_numpy(v).contiguous().to(device) for k, v in d.items()}


def empty_traj_like(tr):
    return {k: torch.zeros_like(v) for k, v in tr.items()}


def alloc_rollout_out(B, n_steps, A, device="cuda", pin=False):
    kw = dict(device=device)
    if pin and device == "cpu":
        kw["pin_memory"] = True
    return dict(overlap=torch.zeros((B, n_steps, A), dtype=torch.uint8, **kw),
                offroad=torch.zeros((B, n_steps, A), dtype=torch.uint8, **kw),
                offroad_dist=torch.zeros((B, n_steps, A), dtype=torch.float32, **kw),
                log_div=torch.zeros((B, n_steps, A), dtype=torch.float32, **kw),
                any_overlap=torch.zeros((B, A), dtype=torch.uint8, **kw),
                any_offroad=torch.zeros((B, A), dtype=torch.uint8, **kw),
                ade=torch.zeros((B, A), dtype=torch.float32, **kw))
