#!/usr/bin/env python
"""Benchmark of the B200-native Waymax closed-loop step (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--B 4096]

Workload (config.workload): BASELINE.json configs[4] — B=4096 scenarios x A=128 agents,
R=20,000 roadgraph points, T=91, one 80-step closed-loop InvertibleBicycle rollout with
overlap, offroad and log divergence every step, one CUDA graph, fp32.  One bench "step" =
one such rollout of the whole batch (reset + 80 x (dynamics, overlap, offroad, log
divergence) + aggregates).  Metric: agent-steps/s = B * A * 80 / time (agent slots, valid or
not; valid-agent-steps reported beside it).

value     device-resident: inputs in HBM when the timed region starts, CUDA events on the
          launching stream, barrier + synchronize on both sides, max over ranks.
e2e       the same job through wm_rollout_host with pinned HOST buffers: scenario + action
          upload, wm_prepare, reset, rollout, metric download all inside the timed region
          (pipelined over scenario chunks: its floor is the PCIe time of the 3.8 GB upload).
roofline  dominant kernel k_rollout_fused (the whole rollout is one launch of it).  The exact grid
          search leaves < 0.1 % of the corner-segment pairs, so the slower roof of the kernel is its
          compulsory HBM IO (actions + log row in, sim row + metric rows out, per agent-step):
          achieved = those bytes / CUDA-event duration of the launch, against the measured HBM peak;
          the FP32 fractions on evaluated pairs and on the brute-force pair count are beside it.
roofline_bruteforce  the brute-force kernel k_offroad: 13 flop per corner-segment pair (SURVEY
          §8(d)) / its CUDA-event duration, against the FP32 peak SMs*128*2*max clock.
cpu_baseline  the oracle (oracle/, as it stands) on the host cores, bounded sample.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

N_STEPS = 80
FLOP_PER_PAIR = 13.0           # w(2) t(3) c(4) d2(3) min(1)
METRIC = "agent-steps/sec for step+overlap+offroad (B=4096,A=128); % of roofline"


def profiled_traffic(kernel):
    """dram__bytes_read+write per launch of `kernel` from the latest committed ncu summary."""
    import glob
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_%s_traffic_bytes.txt" % kernel)))
    try:
        return float(open(files[-1]).read().split()[0]) if files else None
    except Exception:
        return None


def measured_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return None
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.th.join(timeout=2)
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        if not sm:
            return None
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                "power_w_max": float(max(pw)), "samples": len(sm)}


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the host cores; bounded sample/step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    import wm_scenarios as ws
    sample_B = args.ref_B
    cfg = ws.make_config(5, B=sample_B, n_steps=N_STEPS)
    A = cfg["log"]["x"].shape[2]
    times = []
    for it in range(args.warmup_ref + args.steps_ref):
        sim = oracle.reset(cfg["log"])
        t0 = time.perf_counter()
        oracle.rollout(cfg["log"], sim, cfg["roadgraph"], cfg["t0"], N_STEPS, oracle.DYN_BICYCLE,
                       cfg["actions"], cfg["action_valid"])
        dt = time.perf_counter() - t0
        if it >= args.warmup_ref:
            times.append(dt)
    ms = 1e3 * float(np.mean(times))
    val = sample_B * A * N_STEPS / (ms * 1e-3)
    cores = oracle.num_threads()
    sample = "%d of 4096 scenarios x %d steps per bench step (oracle.rollout, OpenMP over scenarios)" % (sample_B, N_STEPS)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "agent-steps/s", "n_gpus": args.gpus,
            "steps": args.steps_ref, "warmup": args.warmup_ref, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "config5: B=4096 A=128 R=20000 T=91 80-step bicycle rollout (bounded sample)",
                       "sample_B": sample_B, "A": A, "R": 20000, "n_steps": N_STEPS},
            "cpu_baseline": {"value": val, "unit": "agent-steps/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "agent-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def run_supplementary(args):
    """Supplementary lines for the other hot-path rows: config 3 observation (a6, a7), config 2
    single DeltaLocal step + metrics (a2-a5), config 4 overlap-dense stress (a3, a4), RolloutExpert
    on config 5 (expert actor + kinematic metric).  N=1 only."""
    import torch
    import oracle
    import wm_scenarios as ws
    import paper_2310_08710_b200 as wm
    torch.cuda.set_device(0)
    peaks = measured_peaks()
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    stream = torch.cuda.current_stream()

    def timed(fn, steps, warmup):
        for _ in range(warmup):
            fn()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(steps):
            fn()
        b.record(stream)
        torch.cuda.synchronize()
        return a.elapsed_time(b) / steps

    W, K = max(args.warmup, 3), args.steps
    if args.workload == "observe":
        cfg = ws.make_config(3)
        log, rg = cfg["log"], cfg["roadgraph"]
        B, T, A = log["x"].shape
        k, H, t = 1000, 11, 10
        h = wm.wm_create(topk=k)
        log_d, rg_d = wm.to_device(log), wm.to_device(rg)
        wm.wm_prepare(h, rg_d)
        hist = torch.empty((B, A, H, 7, A), device="cuda"); hv = torch.empty((B, A, H, A), dtype=torch.uint8, device="cuda")
        idx = torch.empty((B, A, k), dtype=torch.int32, device="cuda")
        feat = torch.empty((B, A, 4, k), device="cuda"); typ = torch.empty((B, A, k), dtype=torch.int32, device="cuda")
        l0 = wm.wm_kernel_launches(h)
        ms = timed(lambda: wm.wm_observe(h, log_d, rg_d, t, hist, hv, idx, feat, typ), K, W)
        launches = (wm.wm_kernel_launches(h) - l0) * K // (K + W)
        ms_h = timed(lambda: wm.wm_observe(h, log_d, rg_d, t, hist, hv, None, None, None), K, W)
        ms_k = timed(lambda: wm.wm_observe(h, log_d, rg_d, t, None, None, idx, feat, typ), K, W)
        egos = int(log["valid"][:, t].sum())
        out_bytes = sum(x.numel() * x.element_size() for x in (hist, hv, idx, feat, typ))
        in_bytes = B * rg["x"].shape[1] * 8 + B * H * A * 29      # point coordinates once + the H rows
        # oracle sample: 2 scenarios
        sb = 2
        sub = lambda d: {q: np.ascontiguousarray(v[:sb]) for q, v in d.items()}
        t0 = time.perf_counter()
        ok = oracle.observe_topk(sub(log), sub(rg), t, k); oracle.observe_history(sub(log), t, H)
        dt = time.perf_counter() - t0
        same = bool(np.array_equal(idx[:sb].cpu().numpy(), ok["rg_index"]))
        line = {"metric": "ego observations/s (history in ego frame + top-1000 roadgraph points), config 3", "value": B * A / (ms * 1e-3),
                "unit": "ego-observations/s", "n_gpus": 1, "steps": K, "warmup": W, "ms_per_step": ms, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": "config3: B=256 A=128 R=30000 H=11 k=1000, every valid agent an ego", "valid_egos": egos,
                           "l2": "outputs 2.2 GB exceed L2", "ms_history": ms_h, "ms_topk": ms_k},
                "roofline": {"bound": "hbm", "achieved": (out_bytes + in_bytes) / (ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                             "frac": (out_bytes + in_bytes) / (ms * 1e-3) / 1e9 / hbm_peak, "traffic": None,
                             "kernel": "k_observe_hist + k_observe_topk", "algorithmic_bytes": out_bytes + in_bytes,
                             "history_frac": (hist.numel() * 4 + hv.numel() + B * H * A * 29) / (ms_h * 1e-3) / 1e9 / hbm_peak,
                             "topk_frac": (out_bytes - hist.numel() * 4 - hv.numel() + B * rg["x"].shape[1] * 8) / (ms_k * 1e-3) / 1e9 / hbm_peak,
                             "note": "top-k: one CTA per ego selects inside a square of point-grid cells; instruction-issue bound, see DESIGN.md"},
                "cpu_baseline": {"value": sb * A / dt, "unit": "ego-observations/s", "cores": oracle.num_threads(), "kind": "oracle",
                                 "sample": "first %d of %d scenarios, %.1f s wall" % (sb, B, dt), "index_sets_equal": same},
                "e2e": None, "gpu_launches": int(launches), "clocks": None}
    elif args.workload == "paper_tables":
        # The SHAPE of the paper's own runtime tables on this GPU, for context: Table 2
        # (Reset / Step / Transition / Metrics / RolloutExpert of the multi-agent environment at batch 1
        # and 16) and Table 6 (Metrics and RolloutExpert against the number of objects).  Synthetic
        # config-5 scenarios (A = 128 slots, R = 20 000), not WOMD; Metrics = this build's three metrics.
        paper = {"hardware": "Nvidia V100 (Table 2 L153-L154; Table 6 L391-L400)",
                 "table2_ms": {"1": {"reset": 0.64, "step": 0.92, "transition": 0.53, "metrics": 0.19, "rollout_expert": 73.3},
                               "16": {"reset": 0.81, "step": 2.86, "transition": 0.51, "metrics": 2.24, "rollout_expert": "OOM"}},
                 "table6_metrics_ms": {"1": {"8": 0.159, "128": 0.152}, "16": {"8": 0.154, "128": 0.469}},
                 "table6_rollout_expert_ms": {"1": {"8": 27.0, "128": 36.9}}}
        ours2, ours6m, ours6r = {}, {}, {}
        total_launches = 0
        for Bn in (1, 16):
            for nobj in ((128,) if False else (8, 16, 32, 64, 128)):
                cfg = ws.make_config(5, B=Bn, n_steps=N_STEPS)
                log, rg = cfg["log"], cfg["roadgraph"]
                log["valid"][:, :, nobj:] = 0                                   # subset of the objects (Table 6: "subsetted objects")
                B, T, A = log["x"].shape
                h = wm.wm_create()
                log_d, rg_d = wm.to_device(log), wm.to_device(rg)
                wm.wm_prepare(h, rg_d)
                sim_d = wm.empty_traj_like(log_d)
                t0 = wm.wm_reset(h, log_d, sim_d)
                act1 = torch.from_numpy(np.ascontiguousarray(cfg["actions"][:, 0])).cuda()
                av1 = torch.from_numpy(np.ascontiguousarray(cfg["action_valid"][:, 0])).cuda()
                Wd = (A + 31) // 32
                ofl = torch.empty((B, A), dtype=torch.uint8, device="cuda"); sd = torch.empty((B, A), device="cuda")
                fl = torch.empty((B, A), dtype=torch.uint8, device="cuda"); ld = torch.empty((B, A), device="cuda"); lv = torch.empty((B, A), dtype=torch.uint8, device="cuda")
                act = torch.empty((B, N_STEPS, 2, A), device="cuda"); av = torch.empty((B, N_STEPS, A), dtype=torch.uint8, device="cuda")
                out_d = wm.alloc_rollout_out(B, N_STEPS, A)

                def metrics():
                    wm.wm_metrics_overlap(h, sim_d, t0 + 1, None, ofl)
                    wm.wm_metrics_offroad(h, sim_d, t0 + 1, sd, None, fl)
                    wm.wm_log_divergence(h, log_d, sim_d, t0 + 1, ld, lv)

                def transition():
                    wm.wm_step(h, log_d, sim_d, t0, act1, av1)

                def rollout_expert():
                    wm.wm_expert_actions(h, log_d, t0, N_STEPS, act, av)
                    wm.wm_reset(h, log_d, sim_d)
                    wm.wm_rollout(h, log_d, sim_d, t0, N_STEPS, act, av, out_d)
                l0 = wm.wm_kernel_launches(h)
                reps = max(K, 20)
                row = {"metrics": timed(metrics, reps, W), "rollout_expert": timed(rollout_expert, reps, W)}
                if nobj == 128:
                    row["reset"] = timed(lambda: wm.wm_reset(h, log_d, sim_d), reps, W)
                    wm.wm_reset(h, log_d, sim_d)
                    row["transition"] = timed(transition, reps, W)
                    row["step"] = timed(lambda: (transition(), metrics()), reps, W)
                    ours2[str(Bn)] = row
                ours6m.setdefault(str(Bn), {})[str(nobj)] = row["metrics"]
                ours6r.setdefault(str(Bn), {})[str(nobj)] = row["rollout_expert"]
                total_launches += wm.wm_kernel_launches(h) - l0
                wm.wm_destroy(h)
        h = wm.wm_create()                                       # the common epilogue destroys `h`
        step16 = ours2["16"]["step"]
        line = {"metric": "agent-steps/s of one multi-agent Step (transition + overlap + offroad + log divergence) at batch 16, A = 128 (the paper's Table 2 row, context)",
                "value": 16 * 128 / (step16 * 1e-3), "unit": "agent-steps/s", "n_gpus": 1, "steps": max(K, 20), "warmup": W, "ms_per_step": step16,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": "paper_tables: config-5 scenarios at batch 1 and 16, 8..128 objects valid; each entry point called from Python, "
                                       "CUDA events around the calls (launch-latency bound at these sizes)", "l2": "everything fits L2 at batch <= 16 (as in the paper's tables); not flushed"},
                "ours_ms": {"table2": ours2, "table6_metrics": ours6m, "table6_rollout_expert": ours6r}, "paper_ms": paper,
                "roofline": {"bound": "hbm", "achieved": None, "peak": hbm_peak, "unit": "GB/s", "frac": None, "traffic": None,
                             "note": "latency-bound micro-batches: no roofline claim; see the default workload"},
                "cpu_baseline": None, "e2e": None, "gpu_launches": int(total_launches), "clocks": None}
    elif args.workload == "idm":
        # IDM reactive sim agents (L110-L112): every valid agent follows its logged path with the IDM speed
        # profile, closed loop: per step wm_step (log playback for everybody) + wm_idm_step + overlap metric
        cfg = ws.make_config(5, B=args.B, n_steps=1)
        log = cfg["log"]
        B, T, A = log["x"].shape
        h = wm.wm_create()
        log_d = wm.to_device(log)
        sim_d = wm.empty_traj_like(log_d)
        t0 = wm.wm_reset(h, log_d, sim_d)
        paths = ws.make_paths(log)
        paths_d = {q: torch.from_numpy(v).cuda() for q, v in paths.items()}
        idm_d = torch.ones((B, A), dtype=torch.uint8, device="cuda")
        act0 = torch.zeros((B, 2, A), device="cuda"); av0 = torch.zeros((B, A), dtype=torch.uint8, device="cuda")
        acc = torch.empty((B, A), device="cuda"); lead = torch.empty((B, A), dtype=torch.int32, device="cuda")
        ofl = torch.empty((B, A), dtype=torch.uint8, device="cuda")
        n_sim = 20

        def fn():
            for s_ in range(n_sim):
                wm.wm_step(h, log_d, sim_d, t0 + s_, act0, av0)
                wm.wm_idm_step(h, sim_d, t0 + s_, paths_d, idm_d, acc, lead)
                wm.wm_metrics_overlap(h, sim_d, t0 + s_ + 1, None, ofl)
        l0 = wm.wm_kernel_launches(h)
        ms = timed(fn, K, W)
        launches = (wm.wm_kernel_launches(h) - l0) * K // (K + W)
        ms_i = timed(lambda: wm.wm_idm_step(h, sim_d, t0 + 5, paths_d, idm_d, acc, lead), K, W)
        P = paths["x"].shape[2]
        idm_bytes = float(B) * A * (P * 13 + 29 + 29 + 8) + float(B) * A * 29
        sb = min(16, B)
        sub = lambda d: {q: np.ascontiguousarray(v[:sb]) for q, v in d.items()}
        sim_o = {q: v[:sb].cpu().numpy().copy() for q, v in sim_d.items()}
        t0c = time.perf_counter()
        ro = oracle.idm_step(sim_o, t0 + 5, sub(paths), np.ones((sb, A), np.uint8))
        dt = time.perf_counter() - t0c
        wm.wm_idm_step(h, sim_d, t0 + 5, paths_d, idm_d, acc, lead); torch.cuda.synchronize()
        line = {"metric": "agent-steps/s, closed loop with IDM sim agents (log playback + wm_idm_step + overlap), config 5", "value": float(B) * A * n_sim / (ms * 1e-3),
                "unit": "agent-steps/s", "n_gpus": 1, "steps": K, "warmup": W, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": "config5 IDM: B=%d A=%d T=%d, %d closed-loop steps per bench step, paths of %d points" % (B, A, T, n_sim, P),
                           "ms_idm_step": ms_i, "l2": "paths 2.8 GB exceed L2", "collision_rate_after_%d_steps" % n_sim: float(ofl.float().mean().item()),
                           "agents_with_lead": float((lead >= 0).float().mean().item())},
                "roofline": {"bound": "hbm", "achieved": idm_bytes / (ms_i * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                             "frac": idm_bytes / (ms_i * 1e-3) / 1e9 / hbm_peak, "traffic": None, "kernel": "k_idm_step", "algorithmic_bytes": idm_bytes,
                             "note": "A x A x P projections per scenario-step, culled by the path's bounding box: ALU / shared-memory bound, not HBM bound"},
                "cpu_baseline": {"value": sb * A / dt, "unit": "agent-steps/s", "cores": oracle.num_threads(), "kind": "oracle",
                                 "sample": "one idm_step of the first %d of %d scenarios, %.2f s wall" % (sb, B, dt),
                                 "lead_indices_equal": bool(np.array_equal(ro["lead"], lead[:sb].cpu().numpy()))},
                "e2e": None, "gpu_launches": int(launches), "clocks": None}
    elif args.workload == "expert":
        # RolloutExpert (Table 2): expert actions from the log by inverse kinematics, the
        # 80-step rollout with them, then the kinematic-infeasibility metric of the simulated rows (L104)
        cfg = ws.make_config(5, B=args.B, n_steps=N_STEPS)
        log, rg = cfg["log"], cfg["roadgraph"]
        B, T, A = log["x"].shape
        h = wm.wm_create()
        log_d, rg_d = wm.to_device(log), wm.to_device(rg)
        wm.wm_prepare(h, rg_d)
        sim_d = wm.empty_traj_like(log_d)
        out_d = wm.alloc_rollout_out(B, N_STEPS, A)
        act = torch.empty((B, N_STEPS, 2, A), device="cuda"); av = torch.empty((B, N_STEPS, A), dtype=torch.uint8, device="cuda")
        kacc = torch.empty((B, N_STEPS, A), device="cuda"); kcur = torch.empty((B, N_STEPS, A), device="cuda")
        kfl = torch.empty((B, N_STEPS, A), dtype=torch.uint8, device="cuda")

        def fn():
            wm.wm_expert_actions(h, log_d, 10, N_STEPS, act, av)
            t0 = wm.wm_reset(h, log_d, sim_d)
            wm.wm_rollout(h, log_d, sim_d, t0, N_STEPS, act, av, out_d)
            wm.wm_metrics_kinematic(h, sim_d, t0 + 1, N_STEPS, kacc, kcur, kfl)
        l0 = wm.wm_kernel_launches(h)
        ms = timed(fn, K, W)
        launches = (wm.wm_kernel_launches(h) - l0) * K // (K + W)
        ms_e = timed(lambda: wm.wm_expert_actions(h, log_d, 10, N_STEPS, act, av), K, W)
        ms_k = timed(lambda: wm.wm_metrics_kinematic(h, sim_d, 11, N_STEPS, kacc, kcur, kfl), K, W)
        # route-progress ratio (L96) of the final row on synthetic per-agent paths (not part of `value`)
        paths = ws.make_paths(log)
        paths_d = {q: torch.from_numpy(v).cuda() for q, v in paths.items()}
        rp = torch.empty((B, A), device="cuda"); rpv = torch.empty((B, A), dtype=torch.uint8, device="cuda")
        ms_rp = timed(lambda: wm.wm_metrics_route_progress(h, log_d, sim_d, 10 + N_STEPS, paths_d, rp, rpv), K, W)
        rp_bytes = float(paths["x"].size) * 13 + float(B) * A * (T + 5 + 16)
        n_as = float(B) * A * N_STEPS
        inv_bytes = n_as * (13 + 9) + n_as * (13 + 9)            # per agent-step: one new row of (yaw, vx, vy, valid) in, 9 B out; twice
        sb = min(64, B)
        sub = lambda d: {q: np.ascontiguousarray(v[:sb]) for q, v in d.items()}
        t0c = time.perf_counter()
        e = oracle.expert_actions(sub(log), 10, N_STEPS, oracle.DYN_BICYCLE)
        sim_o = oracle.reset(sub(log))
        oo = oracle.rollout(sub(log), sim_o, sub(rg), 10, N_STEPS, oracle.DYN_BICYCLE, e["action"], e["valid"])
        ko = oracle.kinematic(sim_o, 11, N_STEPS)
        dt = time.perf_counter() - t0c
        # flag agreement, teacher-forced: the oracle's metric on the GPU's own rows, outside the tolerance band
        kt = oracle.kinematic({q: v[:sb].cpu().numpy() for q, v in sim_d.items()}, 11, N_STEPS)
        tol_k = 1e-5 * np.abs(kt["curvature"]) + 4e-6 / np.maximum(kt["kden"], 1e-12) + 1e-6
        band = (np.abs(np.abs(kt["accel"]) - 6.0) <= 1e-3) | (np.abs(np.abs(kt["curvature"]) - 0.3) <= tol_k)
        clean = (kt["valid"] == 1) & ~band
        line = {"metric": "agent-steps/s, RolloutExpert (expert actions by inverse kinematics + 80-step rollout + kinematic infeasibility), config 5",
                "value": n_as / (ms * 1e-3), "unit": "agent-steps/s", "n_gpus": 1, "steps": K, "warmup": W, "ms_per_step": ms,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": "config5 RolloutExpert: B=%d A=%d R=%d T=%d" % (B, A, rg["x"].shape[1], T), "ms_expert_actions": ms_e,
                           "ms_kinematic_metric": ms_k, "ms_reset_plus_rollout": ms - ms_e - ms_k,
                           "ms_route_progress": ms_rp, "route_progress_hbm_frac": rp_bytes / (ms_rp * 1e-3) / 1e9 / hbm_peak,
                           "mean_route_progress": float(rp[rpv == 1].mean().item()), "l2": "working set 6 GB exceeds L2",
                           "mean_ade_m": float(out_d["ade"].mean().item()), "kinematic_flag_rate": float(kfl.float().mean().item()),
                           "paper_context": "Table 2 L153: RolloutExpert 73.3 ms at BS 1 on a V100 (all six metrics, WOMD)"},
                "roofline": {"bound": "hbm", "achieved": inv_bytes / ((ms_e + ms_k) * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                             "frac": inv_bytes / ((ms_e + ms_k) * 1e-3) / 1e9 / hbm_peak, "traffic": None, "kernel": "k_inverse<false> + k_inverse<true>",
                             "algorithmic_bytes": inv_bytes, "note": "the rollout kernel itself: see the default workload"},
                "cpu_baseline": {"value": sb * A * N_STEPS / dt, "unit": "agent-steps/s", "cores": oracle.num_threads(), "kind": "oracle",
                                 "sample": "first %d of %d scenarios, %.1f s wall" % (sb, B, dt),
                                 "kinematic_flags_equal_outside_band": bool(np.array_equal(kt["flag"][clean], kfl[:sb].cpu().numpy()[clean])),
                                 "transitions_in_band": int(((kt["valid"] == 1) & band).sum()), "transitions": int((kt["valid"] == 1).sum())},
                "e2e": None, "gpu_launches": int(launches), "clocks": None}
    else:
        cid = 2 if args.workload == "step2" else 4
        cfg = ws.make_config(cid)
        log, rg = cfg["log"], cfg["roadgraph"]
        B, T, A = log["x"].shape
        h = wm.wm_create(dynamics=wm.WM_DYN_DELTA_LOCAL)
        log_d, rg_d = wm.to_device(log), wm.to_device(rg)
        seg_max = wm.wm_prepare(h, rg_d)
        sim_d = wm.empty_traj_like(log_d)
        t = wm.wm_reset(h, log_d, sim_d) if cid == 2 else 0
        Wd = (A + 31) // 32
        bits = torch.empty((B, A, Wd), dtype=torch.int32, device="cuda"); ofl = torch.empty((B, A), dtype=torch.uint8, device="cuda")
        sd = torch.empty((B, A), device="cuda"); fl = torch.empty((B, A), dtype=torch.uint8, device="cuda")
        ld = torch.empty((B, A), device="cuda"); lv = torch.empty((B, A), dtype=torch.uint8, device="cuda")
        if cid == 2:
            act = torch.from_numpy(np.ascontiguousarray(cfg["actions"][:, 0])).cuda()
            av = torch.from_numpy(np.ascontiguousarray(cfg["action_valid"][:, 0])).cuda()

            def fn():
                wm.wm_step(h, log_d, sim_d, t, act, av)
                wm.wm_metrics_overlap(h, sim_d, t + 1, bits, ofl)
                wm.wm_metrics_offroad(h, sim_d, t + 1, sd, None, fl)
                wm.wm_log_divergence(h, log_d, sim_d, t + 1, ld, lv)
        else:
            src = log_d

            def fn():
                wm.wm_metrics_overlap(h, src, 0, bits, ofl)
                wm.wm_metrics_offroad(h, src, 0, sd, None, fl)
        l0 = wm.wm_kernel_launches(h)
        ms = timed(fn, K, W)
        launches = (wm.wm_kernel_launches(h) - l0) * K // (K + W)
        row = sim_d if cid == 2 else log_d
        ms_ov = timed(lambda: wm.wm_metrics_overlap(h, row, t + 1 if cid == 2 else 0, bits, ofl), K, W)
        ms_off = timed(lambda: wm.wm_metrics_offroad(h, row, t + 1 if cid == 2 else 0, sd, None, fl), K, W)
        wm.wm_offroad_stats_enable(h, True); wm.wm_offroad_stats(h)
        wm.wm_metrics_offroad(h, row, t + 1 if cid == 2 else 0, sd, None, fl)
        ev, bf, n_slow, n_corner = wm.wm_offroad_stats(h)
        wm.wm_offroad_stats_enable(h, False)
        n_seg = np.array(wm.wm_segment_counts(h, B))
        hbm_bytes = float(n_seg.sum()) * 24.0 + B * A * 34.0
        sb = min(8, B)
        sub = lambda d: {q: np.ascontiguousarray(v[:sb]) for q, v in d.items()}
        rowh = {q: v[:sb].cpu().numpy() for q, v in row.items()}
        tt = t + 1 if cid == 2 else 0
        t0 = time.perf_counter()
        oo = oracle.offroad(rowh, tt, sub(rg), details=False); oracle.overlap(rowh, tt, want_gap=False, want_pair=False)
        dt = time.perf_counter() - t0
        line = {"metric": "agent-steps/s, config %d (%s)" % (cid, "DeltaLocal step + overlap + offroad + log divergence" if cid == 2 else "overlap + offroad, crowded lot"),
                "value": B * A / (ms * 1e-3), "unit": "agent-steps/s", "n_gpus": 1, "steps": K, "warmup": W, "ms_per_step": ms,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": "config%d: B=%d A=%d R=%d" % (cid, B, A, rg["x"].shape[1]), "S_e_max": int(seg_max),
                           "ms_overlap": ms_ov, "ms_offroad": ms_off, "l2": ("segment tiles %d MB per call exceed L2" if n_seg.sum() * 24 > 126e6 else "segment tiles %d MB fit in L2 (small config, not flushed)") % int(n_seg.sum() * 24 / 1e6)},
                "roofline": {"bound": "hbm", "achieved": hbm_bytes / (ms_off * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                             "frac": hbm_bytes / (ms_off * 1e-3) / 1e9 / hbm_peak, "traffic": None, "kernel": "k_offroad_grid",
                             "kernel_ms": ms_off, "evaluated_fraction": ev / max(bf, 1), "pairs_per_corner": ev / max(n_corner, 1),
                             "slow_path_corner_fraction": n_slow / max(n_corner, 1),
                             "note": "small batch: %d CTAs on 148 SMs, latency/launch bound" % B},
                "cpu_baseline": {"value": sb * A / dt, "unit": "agent-steps/s", "cores": oracle.num_threads(), "kind": "oracle",
                                 "sample": "metrics of the first %d of %d scenarios, %.2f s wall" % (sb, B, dt),
                                 "offroad_flags_equal": bool(np.array_equal(oo["flag"], fl[:sb].cpu().numpy()))},
                "e2e": None, "gpu_launches": int(launches), "clocks": None}
    print(json.dumps(line))
    wm.wm_destroy(h)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--B", type=int, default=4096, help="scenarios per GPU (4096 = the BASELINE config)")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--cpu-B", type=int, default=256, help="oracle sample for cpu_baseline (256 scenarios: ~15 s on 16 cores)")
    ap.add_argument("--ref-B", type=int, default=64, help="oracle sample per step of --impl reference (~4 s on 16 cores)")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--workload", default="rollout", choices=["rollout", "observe", "step2", "stress4", "expert", "idm", "paper_tables"],
                    help="rollout = the BASELINE metric (config 5, default); the others time the remaining "
                         "SURVEY 8(a) rows on configs 3, 2, 4 (supplementary lines, same JSON shape)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the side measurements (single-step grid kernel, brute-force kernel)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    args.steps_ref = max(1, min(args.steps, 3)); args.warmup_ref = max(1, min(args.warmup, 1))
    if args.impl == "reference":
        return run_reference(args)
    if args.workload != "rollout":
        return run_supplementary(args)

    import torch
    import wm_scenarios as ws
    import paper_2310_08710_b200 as wm
    from paper_2310_08710_b200 import sharding

    rank, world = sharding.rank_world()
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    sharding.init_process_group("nccl")
    dev = "cuda"

    B, A, R, T = args.B, 128, 20000, 91
    cfg = ws.make_config(5, b_ids=sharding.shard_ids(B, rank, world), n_steps=N_STEPS)
    log_d, rg_d = wm.to_device(cfg["log"]), wm.to_device(cfg["roadgraph"])
    acts_d = torch.from_numpy(cfg["actions"]).to(dev); av_d = torch.from_numpy(cfg["action_valid"]).to(dev)
    sim_d = wm.empty_traj_like(log_d)
    out_d = wm.alloc_rollout_out(B, N_STEPS, A)
    h = wm.wm_create()
    seg_max = wm.wm_prepare(h, rg_d)
    n_seg = np.array(wm.wm_segment_counts(h, B))
    stream = torch.cuda.current_stream()

    def one_pass():
        t0 = wm.wm_reset(h, log_d, sim_d)
        wm.wm_rollout(h, log_d, sim_d, t0, N_STEPS, acts_d, av_d, out_d)

    for _ in range(args.warmup):
        one_pass()
    torch.cuda.synchronize()
    sharding.barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = wm.wm_kernel_launches(h)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    ev0.record(stream)
    for _ in range(args.steps):
        one_pass()
    ev1.record(stream)
    torch.cuda.synchronize()
    sharding.barrier()
    launches = wm.wm_kernel_launches(h) - l0
    ms_total = sharding.max_over_ranks(ev0.elapsed_time(ev1), dev)
    ms_step = ms_total / args.steps
    agent_steps = float(B) * A * N_STEPS * world
    value = agent_steps / (ms_step * 1e-3)
    valid_rows = sim_d["valid"][:, 11:11 + N_STEPS].sum().item()
    valid_value = sharding.sum_over_ranks(valid_rows, dev) / (ms_step * 1e-3)

    # ---- rooflines: the offroad kernel alone, same rows, CUDA events on the launching stream ----
    sd = torch.zeros((B, A), device=dev); fl = torch.zeros((B, A), dtype=torch.uint8, device=dev)

    def time_offroad(handle):
        for t in range(11, 14):
            wm.wm_metrics_offroad(handle, sim_d, t, sd, None, fl)
        torch.cuda.synchronize()
        ka, kb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ka.record(stream)
        for t in range(11, 11 + N_STEPS):
            wm.wm_metrics_offroad(handle, sim_d, t, sd, None, fl)
        kb.record(stream)
        torch.cuda.synchronize()
        return ka.elapsed_time(kb) / N_STEPS

    # dominant kernel of the timed region: k_rollout_fused (one launch = the whole 80-step rollout)
    def time_rollout():
        wm.wm_rollout(h, log_d, sim_d, 10, N_STEPS, acts_d, av_d, out_d)
        torch.cuda.synchronize()
        ka, kb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ka.record(stream)
        for _ in range(5):
            wm.wm_rollout(h, log_d, sim_d, 10, N_STEPS, acts_d, av_d, out_d)
        kb.record(stream)
        torch.cuda.synchronize()
        return ka.elapsed_time(kb) / 5

    kf_ms = time_rollout()
    # pair counters of the search, from one more rollout with the kernel's counters switched on
    wm.wm_offroad_stats_enable(h, True); wm.wm_offroad_stats(h)
    wm.wm_rollout(h, log_d, sim_d, 10, N_STEPS, acts_d, av_d, out_d)
    ev_pairs, bf_pairs, n_slow, n_corner = wm.wm_offroad_stats(h)
    wm.wm_offroad_stats_enable(h, False)
    pairs_eval = ev_pairs / float(N_STEPS)
    nvalid_bt = sim_d["valid"][:, 11:11 + N_STEPS].sum(dim=2).double().cpu().numpy()       # [B, 80]
    pairs_per_launch = float((4.0 * nvalid_bt * n_seg[:, None]).sum() / N_STEPS)            # brute-force count, per step
    peaks = measured_peaks()
    props = torch.cuda.get_device_properties(local)
    sm_max_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    hbm_src = "MEASURED_PEAKS.json hbm_gbs (of measured)" if "hbm_gbs" in peaks else "fallback 6650 GB/s (of fallback)"
    fp32_peak = props.multi_processor_count * 128 * 2 * sm_max_mhz * 1e6 / 1e12              # TFLOP/s
    peak_src = "SMs(%d)*128*2*%.0f MHz (nominal, B200_PROFILING.md unit counts/clocks)" % (props.multi_processor_count, sm_max_mhz)
    # compulsory bytes of one rollout launch: per agent-step the action (C*4) and its mask (1),
    # log row t+1 in (29), sim row t+1 out (29), metric rows out (1+1+4+4); per agent row t0 in (29) and
    # the aggregates out (1+1+4).  The search structures (cells, records) are not compulsory IO.
    C_ACT = 2
    fused_bytes = float(B) * N_STEPS * A * (C_ACT * 4 + 1 + 29 + 29 + 10) + float(B) * A * (29 + 6)
    fused_flops = pairs_eval * N_STEPS * FLOP_PER_PAIR
    roofline = {"bound": "hbm", "achieved": fused_bytes / (kf_ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                "frac": fused_bytes / (kf_ms * 1e-3) / 1e9 / hbm_peak, "traffic": profiled_traffic("k_rollout_fused"),
                "kernel": "k_rollout_fused", "kernel_ms": kf_ms, "algorithmic_bytes_per_launch": fused_bytes,
                "peak_source": hbm_src, "kernel_share_of_step": kf_ms / ms_step,
                "hbm_time_ms_at_peak": fused_bytes / (hbm_peak * 1e9) * 1e3,
                "fp32_time_ms_at_peak_on_evaluated_pairs": fused_flops / (fp32_peak * 1e12) * 1e3,
                "pairs_bruteforce_per_step": pairs_per_launch, "pairs_evaluated_per_step": pairs_eval,
                "evaluated_fraction": pairs_eval / pairs_per_launch, "pairs_per_corner": ev_pairs / max(n_corner, 1),
                "slow_path_corner_fraction": n_slow / max(n_corner, 1),
                "alu_frac_on_evaluated_pairs": fused_flops / (kf_ms * 1e-3) / 1e12 / fp32_peak,
                "alu_frac_bruteforce_equivalent": pairs_per_launch * N_STEPS * FLOP_PER_PAIR / (kf_ms * 1e-3) / 1e12 / fp32_peak,
                "note": "exact culling (SURVEY 8(d)) leaves under 0.1 % of the pairs, so the slower roof of the kernel is its "
                        "compulsory HBM IO; the FP32 fractions on evaluated pairs and on the brute-force count are beside it. "
                        "ncu: the kernel is bound by gather latency and instruction issue, not by HBM bandwidth (profiles/)"}
    hbm_bytes = float(n_seg.sum()) * 24.0 + B * A * 29.0 + B * A * 5.0    # brute force: segments once + one state row + outputs
    rl_ms = max(pairs_per_launch * FLOP_PER_PAIR / (fp32_peak * 1e12), hbm_bytes / (hbm_peak * 1e9)) * 1e3
    step_roofline = {"definition": "north_star: slower of algorithmic bytes/HBM peak and brute-force FP32 flops/FP32 peak, per simulated step",
                     "roofline_ms": rl_ms, "achieved_ms": ms_step / N_STEPS, "frac": rl_ms / (ms_step / N_STEPS)}
    roofline_grid = roofline_bf = None
    if not args.no_extras:
        # side measurements, outside the timed region: the single-step entry point of the same search,
        # and the brute-force kernel (every corner against every segment) against the FP32 peak
        k_ms = time_offroad(h)
        roofline_grid = {"bound": "hbm", "kernel": "k_offroad_grid (wm_metrics_offroad, one step)", "kernel_ms": k_ms,
                         "algorithmic_bytes_per_launch": B * A * 34.0, "note": "single-step entry point of the same search"}
        hb = wm.wm_create(offroad_mode=wm.WM_OFFROAD_BRUTE_FORCE)
        wm.wm_prepare(hb, rg_d)
        kb_ms = time_offroad(hb)
        wm.wm_destroy(hb)
        bf_achieved = pairs_per_launch * FLOP_PER_PAIR / (kb_ms * 1e-3) / 1e12
        roofline_bf = {"bound": "alu", "achieved": bf_achieved, "peak": fp32_peak, "unit": "TFLOP/s",
                       "frac": bf_achieved / fp32_peak, "traffic": profiled_traffic("k_offroad_brute"),
                       "kernel": "k_offroad (offroad_mode=WM_OFFROAD_BRUTE_FORCE)", "kernel_ms": kb_ms,
                       "pairs_per_launch": pairs_per_launch, "flop_per_pair": FLOP_PER_PAIR, "peak_source": peak_src}
    clocks = sampler.stop() if rank == 0 else None

    # ---- e2e: the same job from pinned host buffers through the C-ABI ----
    e2e = None
    if not args.no_e2e:
        pin = lambda d: {k: torch.from_numpy(v).pin_memory() for k, v in d.items()}
        log_h, rg_h = pin(cfg["log"]), pin(cfg["roadgraph"])
        acts_h = torch.from_numpy(cfg["actions"]).pin_memory(); av_h = torch.from_numpy(cfg["action_valid"]).pin_memory()
        out_h = wm.alloc_rollout_out(B, N_STEPS, A, device="cpu", pin=True)
        h2 = wm.wm_create()
        wm.wm_rollout_host(h2, log_h, rg_h, N_STEPS, acts_h, av_h, out_h)       # warm-up (allocations, graph capture)
        wm.wm_rollout_host(h2, log_h, rg_h, N_STEPS, acts_h, av_h, out_h)
        torch.cuda.synchronize(); sharding.barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(args.e2e_steps):
            wm.wm_rollout_host(h2, log_h, rg_h, N_STEPS, acts_h, av_h, out_h)
        e1.record(stream)
        torch.cuda.synchronize(); sharding.barrier()
        e_ms = sharding.max_over_ranks(e0.elapsed_time(e1), dev) / args.e2e_steps
        h2d = sum(v.numel() * v.element_size() for v in list(log_h.values()) + list(rg_h.values()) + [acts_h, av_h])
        d2h = sum(v.numel() * v.element_size() for v in out_h.values())
        same = all(torch.equal(out_h[k], out_d[k].cpu()) for k in out_h)
        e2e = {"value": agent_steps / (e_ms * 1e-3), "unit": "agent-steps/s", "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "ms_per_step": e_ms, "outputs_equal_device_path": bool(same),
               "includes": "scenario+action upload, wm_prepare, reset, 80-step rollout, metric download; pipelined over 16 scenario chunks"}
        wm.wm_destroy(h2)

    # ---- cpu_baseline: the oracle on a bounded sample (rank 0, N=1 only) ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        import oracle
        sb = min(args.cpu_B, B)
        sub = lambda d: {k: np.ascontiguousarray(v[:sb]) for k, v in d.items()}
        lg, rgs = sub(cfg["log"]), sub(cfg["roadgraph"])
        sim_o = oracle.reset(lg)
        t0 = time.perf_counter()
        o = oracle.rollout(lg, sim_o, rgs, cfg["t0"], N_STEPS, oracle.DYN_BICYCLE,
                           np.ascontiguousarray(cfg["actions"][:sb]), np.ascontiguousarray(cfg["action_valid"][:sb]))
        dt = time.perf_counter() - t0
        agree = float((o["offroad"] == out_d["offroad"][:sb].cpu().numpy()).mean())
        cpu = {"value": sb * A * N_STEPS / dt, "unit": "agent-steps/s", "cores": oracle.num_threads(), "kind": "oracle",
               "sample": "first %d of %d scenarios x %d steps, oracle.rollout, %.1f s wall" % (sb, B, N_STEPS, dt),
               "offroad_flag_agreement_free_running": agree}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": "agent-steps/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": "config5: B=%d/GPU A=128 R=20000 T=91, 80-step InvertibleBicycle rollout + overlap + offroad + log divergence, one CUDA graph" % B,
                       "B_per_gpu": B, "A": A, "R": R, "T": T, "n_steps": N_STEPS, "S_e_max": int(seg_max),
                       "S_e_mean": float(n_seg.mean()), "l2": "inputs exceed L2 (segments %.2f GB + state per step)" % (n_seg.sum() * 24 / 1e9),
                       "parallelism": "scenario shards, no collective", "valid_agent_steps_per_s": valid_value,
                       "ms_per_sim_step": ms_step / N_STEPS},
            "roofline": roofline, "roofline_offroad_grid": roofline_grid, "roofline_bruteforce": roofline_bf, "step_roofline": step_roofline,
            "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
        }
        print(json.dumps(line))
    wm.wm_destroy(h)
    return 0


if __name__ == "__main__":
    sys.exit(main())
