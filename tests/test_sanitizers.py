"""CPU (-m "not gpu"): the oracle under AddressSanitizer + UndefinedBehaviorSanitizer.

Every parity claim rests on oracle/wm_oracle.cpp, a C++ file that indexes raw arrays handed over by ctypes.  An
out-of-bounds read there would not crash; it would quietly change an expected value.  This test builds the same source
with -fsanitize=address,undefined and drives every oracle entry point on config-1-sized inputs (ragged shapes, holes in
the validity masks, fewer valid points than k) in a child process with libasan preloaded.  Any report fails the test.
"""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

DRIVER = r"""
import numpy as np
import oracle, wm_scenarios as ws
cfg = ws.make_config(1, n_steps=12)
log, rg = cfg["log"], cfg["roadgraph"]
B, T, A = log["x"].shape
rg["valid"][:, 5::13] = 0                                   # holes: broken polylines, isolated road-edge points
sim = oracle.reset(log)
t0, n = cfg["t0"], 12
acts, av = np.ascontiguousarray(cfg["actions"][:, :n]), np.ascontiguousarray(cfg["action_valid"][:, :n])
out = oracle.rollout(log, sim, rg, t0, n, oracle.DYN_BICYCLE, acts, av)
assert out["offroad"].shape == (B, n, A)
for dyn, C in ((oracle.DYN_DELTA_LOCAL, 3), (oracle.DYN_DELTA_GLOBAL, 3)):
    s2 = oracle.reset(log)
    oracle.step(log, s2, t0, dyn, np.zeros((B, C, A), np.float32), np.ones((B, A), np.uint8))
oracle.overlap(sim, t0 + n); oracle.offroad(sim, t0 + n, rg); oracle.log_divergence(log, sim, t0 + n)
[oracle.count_segments(rg, b) for b in range(B)]
oracle.observe_history(sim, t0 + n, 11)
for k, order in ((1, 0), (64, 1), (rg["x"].shape[1], 0)):   # k = R: more than the valid points
    oracle.observe_topk(sim, rg, t0 + n, k, order)
e = oracle.expert_actions(log, 0, T - 1, oracle.DYN_BICYCLE)
oracle.expert_actions(log, 3, 5, oracle.DYN_DELTA_LOCAL)
oracle.kinematic(sim, 1, T - 1)
paths = ws.make_paths(log)
paths["valid"][:, ::3, 7] = 0
oracle.route_progress(log, sim, t0 + n, paths)
oracle.offroute(sim, t0 + n, paths, None, 5.0, 1.0); oracle.offroute(sim, t0 + n, paths, paths, 5.0, 1.0)
oracle.idm_step(oracle.copy_traj(sim), t0, paths, np.ones((B, A), np.uint8))
g = np.ones((B, n, 5, A), np.float32)
oracle.rollout_vjp(sim, t0, n, oracle.DYN_BICYCLE, acts, av, g)
d = oracle.discretize_actions(acts.reshape(B * n, 2, A), [13, 9], [-6.0, -0.3], [6.0, 0.3], av.reshape(B * n, A))
oracle.actions_from_index(d["index"], 2, [13, 9], [-6.0, -0.3], [6.0, 0.3])
print("SAN_OK", oracle.num_threads())
"""


def test_oracle_runs_clean_under_asan_and_ubsan(tmp_path):
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], stdout=subprocess.PIPE, text=True).stdout.strip()
    if not os.path.isabs(asan) or not os.path.exists(asan):
        pytest.skip("this toolchain has no libasan")
    lib = str(tmp_path / "libwm_oracle_san.so")
    subprocess.check_call(["g++", "-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined",
                           "-fno-sanitize-recover=undefined", "-fopenmp", "-ffp-contract=off", "-std=c++17", "-shared", "-fPIC",
                           "-o", lib, os.path.join(ROOT, "oracle", "wm_oracle.cpp")])
    env = dict(os.environ, LD_PRELOAD=os.path.realpath(asan), WM_ORACLE_LIB=lib, PYTHONPATH=ROOT, OMP_NUM_THREADS="2",
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=0:exitcode=97", UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1:exitcode=98")
    res = subprocess.run([sys.executable, "-c", DRIVER], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, timeout=600, cwd=ROOT)
    tail = res.stderr[-3000:]
    assert "AddressSanitizer" not in res.stderr and "runtime error" not in res.stderr, tail
    assert res.returncode == 0 and "SAN_OK" in res.stdout, (res.returncode, tail)
