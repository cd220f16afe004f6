"""-m gpu: wm_observe_topk_static, the entry point for callers that may not allocate device memory.

Who needs it: a simulator step called from inside a job whose framework allocator already owns nearly all
of the GPU's memory (a library's own cudaMalloc then fails or steals the pool's head-room), a planner with
a memory budget frozen at start-up, a latency-critical loop that cannot take cudaMalloc's device-wide
stall.  The entry point takes no handle and keeps its scratch (the bucketed roadgraph points) in an array
built into the library, shared by all calls on a GPU and never cleared.

What is checked: its outputs against the regular, allocating route (wm_create -> wm_prepare -> wm_observe)
on TWO CALLS IN A ROW with different shapes, so the second call runs on the leftovers of the first and the
third on the leftovers of the second; that the driver's free-memory figure does not move across such
calls; that problems beyond the built-in capacity are refused before anything is launched.  The regular
route is itself compared with the oracle in test_gpu_observe.py; both routes run the same kernels, so the
tolerance here is that file's (integers exact, features rtol 1e-5 / atol 2e-4) and in fact the results
are equal bit for bit, which is asserted too since wm.h promises it.

The file is named to be collected last: with `pytest -x` a failure here cannot hide another test.  It
passes alone in a fresh process (the static call is then the first thing the library does on the device)
and after the rest of the suite.
"""
import numpy as np
import pytest
import torch

import wm_scenarios as ws
import paper_2310_08710_b200 as wm
from gpu_util import dev

pytestmark = pytest.mark.gpu


def _outputs(B, A, k):
    return (torch.full((B, A, k), 77, dtype=torch.int32, device="cuda"),
            torch.full((B, A, 4, k), 5.0, device="cuda"),
            torch.full((B, A, k), 77, dtype=torch.int32, device="cuda"))


def _regular(log_d, rg_d, t, k, order):
    """The existing path: a handle, wm_prepare (cudaMalloc inside), wm_observe."""
    B, T, A = log_d["x"].shape
    h = wm.wm_create(topk=k, topk_order=order)
    wm.wm_prepare(h, rg_d)
    out = _outputs(B, A, k)
    wm.wm_observe(h, log_d, rg_d, t, None, None, *out)
    torch.cuda.synchronize()
    wm.wm_destroy(h)
    return out


def _same(got, ref, what):
    for g, r, name in zip(got, ref, ("rg_index", "rg_feat", "rg_type")):
        g, r = g.cpu().numpy(), r.cpu().numpy()
        if g.dtype == np.float32:
            assert np.allclose(g, r, rtol=1e-5, atol=2e-4), (what, name)
        assert np.array_equal(g, r), (what, name, "not bit-equal to wm_prepare + wm_observe")


def test_static_topk_equals_the_allocating_path_on_calls_in_a_row():
    # case 1: two scenarios of config 3 (30 000 points, k = 1000), ascending-index order;
    # case 2: config 1 (4 scenarios, fewer points, another A), k = 64, nearest first, a later row
    c1, c2 = ws.make_config(3, B=2), ws.make_config(1)
    l1, g1 = dev(c1["log"]), dev(c1["roadgraph"])
    l2, g2 = dev(c2["log"]), dev(c2["roadgraph"])
    (B1, _, A1), (B2, _, A2) = l1["x"].shape, l2["x"].shape
    assert g1["x"].shape[1] != g2["x"].shape[1] and B1 != B2
    o1, o2, o3 = _outputs(B1, A1, 1000), _outputs(B2, A2, 64), _outputs(B1, A1, 1000)
    # three calls back to back on one stream, no synchronisation between them: the stream orders them
    wm.wm_observe_topk_static(l1, g1, 10, 1000, *o1)
    wm.wm_observe_topk_static(l2, g2, 40, 64, *o2, topk_order=wm.WM_TOPK_BY_DISTANCE)
    wm.wm_observe_topk_static(l1, g1, 10, 1000, *o3)
    torch.cuda.synchronize()
    r1 = _regular(l1, g1, 10, 1000, wm.WM_TOPK_BY_INDEX)
    r2 = _regular(l2, g2, 40, 64, wm.WM_TOPK_BY_DISTANCE)
    _same(o1, r1, "first call")
    _same(o2, r2, "second call, on the first call's leftovers")
    _same(o3, r1, "third call, on the second call's leftovers")
    v = c1["log"]["valid"][:, 10] == 1
    assert (o1[0].cpu().numpy()[v] >= 0).all()               # something was selected: not a comparison of two empty results

    # no device memory is taken by further calls (kernels are loaded by now, outputs exist already)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        wm.wm_observe_topk_static(l1, g1, 10, 1000, *o1)
        wm.wm_observe_topk_static(l2, g2, 40, 64, *o2, topk_order=wm.WM_TOPK_BY_DISTANCE)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0, "device memory shrank by %d bytes across calls that must not allocate" % (free0 - free1)
    _same(o1, r1, "repeat")
    _same(o2, r2, "repeat")


def test_static_topk_refuses_what_does_not_fit_its_array():
    def problem(B, R, A=2, T=2):
        tr = {k: torch.zeros((B, T, A), device="cuda") for k in wm.TRAJ_F}
        tr["valid"] = torch.ones((B, T, A), dtype=torch.uint8, device="cuda")
        rg = {k: torch.zeros((B, R), device="cuda") for k in wm.RG_F}
        rg.update(type=torch.ones((B, R), dtype=torch.int32, device="cuda"), id=torch.zeros((B, R), dtype=torch.int32, device="cuda"),
                  valid=torch.ones((B, R), dtype=torch.uint8, device="cuda"))
        return tr, rg
    for B, R in ((wm.WM_STATIC_MAX_B + 1, 16), (2, wm.WM_STATIC_MAX_POINTS // 2 + 1)):
        tr, rg = problem(B, R)
        out = _outputs(B, 2, 4)
        with pytest.raises(wm.WmError, match="WM_ERR_TOO_LARGE"):
            wm.wm_observe_topk_static(tr, rg, 0, 4, *out)
        torch.cuda.synchronize()
        assert (out[0] == 77).all() and (out[2] == 77).all()      # nothing was launched
    # the largest shapes that do fit run
    tr, rg = problem(wm.WM_STATIC_MAX_B, wm.WM_STATIC_MAX_POINTS // wm.WM_STATIC_MAX_B)
    out = _outputs(wm.WM_STATIC_MAX_B, 2, 4)
    wm.wm_observe_topk_static(tr, rg, 0, 4, *out)
    torch.cuda.synchronize()
    assert (out[0].cpu().numpy() == np.arange(4)).all()           # all points coincide with the ego: ties -> lower index
