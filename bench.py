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
roofline  the rollout graph = k_rollout_dyn(_bulk) + k_rollout_metrics (one launch of each per 80-step rollout).  The
          exact grid search leaves ~0.1 % of the corner-segment pairs, so the slower roof of the graph is its
          compulsory HBM IO (actions + log row in, sim row + metric rows out, per agent-step):
          achieved = those bytes / CUDA-event duration of the two launches, against the measured HBM peak;
          roofline.kernels has each kernel's own time, bytes and fraction; the FP32 fractions on evaluated
          pairs and on the brute-force pair count are beside it.
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


def source_hash():
    """sha256 over the CUDA sources of the library: ties a profiled number to the code it was taken from."""
    import glob
    import hashlib
    hsh = hashlib.sha256()
    for f in sorted(glob.glob(os.path.join(ROOT, "paper_2310_08710_b200", "csrc", "*.cu*"))):
        hsh.update(open(f, "rb").read())
    return hsh.hexdigest()


TRAFFIC_FILE = os.path.join(ROOT, "profiles", "r03_traffic.json.txt")


def profiled_traffic(kernel):
    """dram__bytes_read + write per launch of `kernel` from the committed ncu pass (profiles/r03_traffic.json.txt,
    written by `bench.py --write-traffic <ncu csv>`).  A number taken from other sources than the ones
    that are being timed is not reported: (None, why)."""
    try:
        d = json.load(open(TRAFFIC_FILE))
    except Exception:
        return None, "no profiles/r03_traffic.json.txt"
    if d.get("source_sha256") != source_hash():
        return None, "profiles/r03_traffic.json.txt was taken from other kernel sources (sha256 differs): re-run the ncu pass"
    v = d.get("kernels", {}).get(kernel)
    return (float(v), "profiles/r03_traffic.json.txt (%s)" % d.get("command", "ncu")) if v is not None else (None, "kernel not in profiles/r03_traffic.json.txt")


def write_traffic(csv_path):
    """Parse `ncu --metrics dram__bytes_read.sum,dram__bytes_write.sum --csv` output into profiles/r03_traffic.json.txt."""
    import csv
    rows = list(csv.reader(open(csv_path)))
    i = [k for k, r in enumerate(rows) if r and r[0] == "ID"][0]
    hdr = rows[i]
    kn, mn, mv, mu = hdr.index("Kernel Name"), hdr.index("Metric Name"), hdr.index("Metric Value"), hdr.index("Metric Unit")
    acc = {}
    for r in rows[i + 1:]:
        if len(r) <= mv or not r[mn].startswith("dram__bytes"):
            continue
        name = r[kn].split("(")[0].split("<")[0].replace("void ", "").strip()
        scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(r[mu], 1.0)
        a = acc.setdefault(name, {})
        a.setdefault(r[0], 0.0)
        a[r[0]] += float(r[mv].replace(",", "")) * scale
    kernels = {k: float(np.mean(list(v.values()))) for k, v in acc.items()}
    out = {"source_sha256": source_hash(), "kernels": kernels, "unit": "bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum)",
           "command": "ncu --metrics dram__bytes_read.sum,dram__bytes_write.sum --clock-control none -c 400 --csv --log-file <csv> python bench.py --steps 2 --warmup 1 --no-cpu --no-e2e --no-extras; python bench.py --write-traffic <csv>"}
    json.dump(out, open(TRAFFIC_FILE, "w"), indent=1)
    print(json.dumps(out))
    return 0


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


def other_configs(wm, ws, torch, hbm_peak, log5_d, sim5_d, stream):
    """The remaining SURVEY 8(a)/(f) rows in the default line: configs 3, 2, 4 (BASELINE.json configs[2], [1], [3]),
    the expert actor / kinematic metric and the IDM step on config-5 scenarios.  Device-resident, CUDA events per
    repetition on the launching stream, L2 flushed (a 256 MB write) before every repetition, 3 warm-ups + 5 timed."""
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def timed(fn, reps=5, warm=3):
        for _ in range(warm):
            fn()
        tot = 0.0
        for _ in range(reps):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream); fn(); b.record(stream)
            torch.cuda.synchronize()
            tot += a.elapsed_time(b)
        return tot / reps

    def rl(nbytes, ms):
        return {"ms": ms, "algorithmic_bytes": float(nbytes), "hbm_frac": nbytes / (ms * 1e-3) / 1e9 / hbm_peak}
    out = {"protocol": "L2 flushed (256 MB write) before every repetition; CUDA events on the launching stream; 3 warm-ups + 5 timed"}
    # ---- config 3: observation (a6, a7) ----
    cfg = ws.make_config(3)
    log, rg = cfg["log"], cfg["roadgraph"]
    B, T, A = log["x"].shape
    R = rg["x"].shape[1]
    k, H, t = 1000, 11, 10
    h = wm.wm_create(topk=k)
    log_d, rg_d = wm.to_device(log), wm.to_device(rg)
    wm.wm_prepare(h, rg_d)
    hist = torch.empty((B, A, H, 7, A), device="cuda"); hv = torch.empty((B, A, H, A), dtype=torch.uint8, device="cuda")
    idx = torch.empty((B, A, k), dtype=torch.int32, device="cuda"); feat = torch.empty((B, A, 4, k), device="cuda")
    typ = torch.empty((B, A, k), dtype=torch.int32, device="cuda")
    l0 = wm.wm_kernel_launches(h)
    ms_h = timed(lambda: wm.wm_observe(h, log_d, rg_d, t, hist, hv, None, None, None))
    ms_k = timed(lambda: wm.wm_observe(h, log_d, rg_d, t, None, None, idx, feat, typ))
    b_h = hist.numel() * 4 + hv.numel() + B * H * A * 29
    b_k = idx.numel() * 4 + feat.numel() * 4 + typ.numel() * 4 + B * R * 8
    out["config3_observe"] = {"workload": "B=%d A=%d R=%d H=%d k=%d, every valid agent an ego" % (B, A, R, H, k),
                              "k_observe_hist": rl(b_h, ms_h), "k_observe_topk": rl(b_k, ms_k), "ms": ms_h + ms_k,
                              "ego_observations_per_s": B * A / ((ms_h + ms_k) * 1e-3)}
    launches = wm.wm_kernel_launches(h) - l0
    wm.wm_destroy(h)
    del hist, hv, idx, feat, typ, log_d, rg_d
    # ---- config 2: one DeltaLocal step + overlap + offroad + log divergence (a2-a5) ----
    for cid in (2, 4):
        cfg = ws.make_config(cid)
        log, rg = cfg["log"], cfg["roadgraph"]
        B, T, A = log["x"].shape
        h = wm.wm_create(dynamics=wm.WM_DYN_DELTA_LOCAL)
        log_d, rg_d = wm.to_device(log), wm.to_device(rg)
        wm.wm_prepare(h, rg_d)
        sim_d = wm.empty_traj_like(log_d)
        Wd = (A + 31) // 32
        bits = torch.empty((B, A, Wd), dtype=torch.int32, device="cuda"); ofl = torch.empty((B, A), dtype=torch.uint8, device="cuda")
        sd = torch.empty((B, A), device="cuda"); fl = torch.empty((B, A), dtype=torch.uint8, device="cuda")
        ld = torch.empty((B, A), device="cuda"); lv = torch.empty((B, A), dtype=torch.uint8, device="cuda")
        l0 = wm.wm_kernel_launches(h)
        if cid == 2:
            t = wm.wm_reset(h, log_d, sim_d)
            act = torch.from_numpy(np.ascontiguousarray(cfg["actions"][:, 0])).cuda()
            av = torch.from_numpy(np.ascontiguousarray(cfg["action_valid"][:, 0])).cuda()
            ms_st = timed(lambda: wm.wm_step(h, log_d, sim_d, t, act, av))
            ms_ov = timed(lambda: wm.wm_metrics_overlap(h, sim_d, t + 1, bits, ofl))
            ms_of = timed(lambda: wm.wm_metrics_offroad(h, sim_d, t + 1, sd, None, fl))
            ms_ld = timed(lambda: wm.wm_log_divergence(h, log_d, sim_d, t + 1, ld, lv))
            n = float(B) * A
            out["config2_step"] = {"workload": "B=%d A=%d R=%d, DeltaLocal step + overlap matrix + offroad + log divergence" % (B, A, rg["x"].shape[1]),
                                   "k_step": rl(n * (29 + 13 + 29 + 29), ms_st), "k_overlap": rl(n * (29 + 4 * Wd + 1), ms_ov),
                                   "k_offroad_grid": rl(n * (29 + 5), ms_of), "k_logdiv": rl(n * (18 + 5), ms_ld),
                                   "ms": ms_st + ms_ov + ms_of + ms_ld, "agent_steps_per_s": n / ((ms_st + ms_ov + ms_of + ms_ld) * 1e-3),
                                   "note": "%d agents per call: launch / latency bound, the HBM fractions are not roofline claims" % int(n)}
        else:
            ms_ov = timed(lambda: wm.wm_metrics_overlap(h, log_d, 0, bits, ofl))
            ms_of = timed(lambda: wm.wm_metrics_offroad(h, log_d, 0, sd, None, fl))
            n = float(B) * A
            gs = wm.wm_grid_stats(h)
            out["config4_stress"] = {"workload": "B=%d A=%d R=%d, overlap matrix + offroad of the crowded lot" % (B, A, rg["x"].shape[1]),
                                     "grid_cells_without_list_frac": {k: v[2] for k, v in gs.items()},
                                     "k_overlap": rl(n * (29 + 4 * Wd + 1), ms_ov), "k_offroad_grid": rl(n * (29 + 5), ms_of),
                                     "ms": ms_ov + ms_of, "pair_tests_per_s": B * A * (A - 1) / 2 / (ms_ov * 1e-3),
                                     "note": "%d agents per call: launch / latency bound, the HBM fractions are not roofline claims" % int(n)}
        launches += wm.wm_kernel_launches(h) - l0
        wm.wm_destroy(h)
        del log_d, rg_d, sim_d
    # ---- expert actor + kinematic metric (NEXT(1)) and the backward pass (NEXT(4)) on the config-5 batch ----
    B, T, A = log5_d["x"].shape
    h = wm.wm_create()
    act = torch.empty((B, N_STEPS, 2, A), device="cuda"); av = torch.empty((B, N_STEPS, A), dtype=torch.uint8, device="cuda")
    kacc = torch.empty((B, N_STEPS, A), device="cuda"); kcur = torch.empty((B, N_STEPS, A), device="cuda")
    kfl = torch.empty((B, N_STEPS, A), dtype=torch.uint8, device="cuda")
    l0 = wm.wm_kernel_launches(h)
    ms_e = timed(lambda: wm.wm_expert_actions(h, log5_d, 10, N_STEPS, act, av))
    ms_m = timed(lambda: wm.wm_metrics_kinematic(h, sim5_d, 11, N_STEPS, kacc, kcur, kfl))
    n_as = float(B) * A * N_STEPS
    g_rows = torch.ones((B, N_STEPS, 5, A), device="cuda"); g_act = torch.empty((B, N_STEPS, 2, A), device="cuda")
    ms_v = timed(lambda: wm.wm_rollout_vjp(h, sim5_d, 10, N_STEPS, act, av, g_rows, g_act, None))
    out["config5_expert"] = {"workload": "B=%d A=%d, 80 transitions per agent" % (B, A), "k_inverse_expert": rl(n_as * 22, ms_e),
                             "k_inverse_kinematic": rl(n_as * 22, ms_m), "k_rollout_vjp": rl(n_as * (13 + 9 + 20 + 8), ms_v)}
    del g_rows, g_act, kacc, kcur, kfl
    # ---- IDM sim agent step (NEXT(2)) on the first 1024 config-5 scenarios ----
    Bi = min(1024, B)
    logi = {q: v[:Bi].contiguous() for q, v in log5_d.items()}
    simi = wm.empty_traj_like(logi)
    t0 = wm.wm_reset(h, logi, simi)
    paths = ws.make_paths({q: v.cpu().numpy() for q, v in logi.items()})
    paths_d = {q: torch.from_numpy(v).cuda() for q, v in paths.items()}
    idm_d = torch.ones((Bi, A), dtype=torch.uint8, device="cuda")
    acc = torch.empty((Bi, A), device="cuda"); lead = torch.empty((Bi, A), dtype=torch.int32, device="cuda")
    ms_i = timed(lambda: wm.wm_idm_step(h, simi, t0, paths_d, idm_d, acc, lead))
    P = paths["x"].shape[2]
    out["config5_idm"] = {"workload": "B=%d A=%d, paths of %d points, every valid agent IDM-controlled" % (Bi, A, P),
                          "k_idm_step": rl(float(Bi) * A * (P * 13 + 29 + 29 + 8), ms_i), "agent_steps_per_s": Bi * A / (ms_i * 1e-3)}
    launches += wm.wm_kernel_launches(h) - l0
    wm.wm_destroy(h)
    return out, int(launches)


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
    ap.add_argument("--no-extras", action="store_true", help="skip the side measurements (single-step grid kernel, brute-force kernel, other configs)")
    ap.add_argument("--write-traffic", default=None, metavar="NCU_CSV", help="parse an ncu dram__bytes csv into profiles/r03_traffic.json.txt and exit")
    args = ap.parse_args()
    if args.write_traffic:
        return write_traffic(args.write_traffic)
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

    # the rollout's two kernels (one graph; the whole 80-step rollout = one launch of each), timed one by one
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
    kt = np.array([wm.wm_rollout_kernel_times(h, log_d, sim_d, 10, N_STEPS, acts_d, av_d, out_d) for _ in range(6)][1:])
    dyn_ms, met_ms = float(kt[:, 0].mean()), float(kt[:, 1].mean())
    # wm_prepare (the static precompute a NEW batch of scenarios needs before its first rollout), and reset alone
    def time_prepare(reps=3):
        wm.wm_prepare(h, rg_d)
        torch.cuda.synchronize()
        ka, kb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ka.record(stream)
        for _ in range(reps):
            wm.wm_prepare(h, rg_d)
        kb.record(stream)
        torch.cuda.synchronize()
        return ka.elapsed_time(kb) / reps
    prepare_ms = sharding.max_over_ranks(time_prepare(), dev)
    grid_stats = wm.wm_grid_stats(h)          # cells per level and how many of them have no candidate list
    ka, kb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ka.record(stream)
    for _ in range(5):
        wm.wm_reset(h, log_d, sim_d)
    kb.record(stream)
    torch.cuda.synchronize()
    reset_ms = ka.elapsed_time(kb) / 5
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
    # FP32 peak as a register-resident FMA loop reaches it in THIS run: scalar FFMA and packed FFMA2
    fp32_measured = {}
    for packed, name in ((0, "ffma"), (1, "ffma2")):
        best = 0.0
        for _ in range(3):
            ms_f, flop = wm.wm_selftest_ffma(h, packed, props.multi_processor_count * 8, 4096)
            best = max(best, flop / (ms_f * 1e-3) / 1e12)
        fp32_measured[name] = best
    fp32_peak_measured = max(fp32_measured.values())
    # Compulsory bytes of the rollout: per agent-step the action (C*4) and its mask (1), log row
    # t+1 in (29), sim row t+1 out (29), metric rows out (1+1+4+4); per agent row t0 in (29) and the
    # aggregates out (1+1+4).  NOT compulsory, hence not counted: the search structures (cells, records) and
    # the metrics kernel's re-read of the simulated rows (21 B per agent-step: x, y, yaw, length, width, valid).
    C_ACT = 2
    n_as = float(B) * N_STEPS * A
    fused_bytes = n_as * (C_ACT * 4 + 1 + 29 + 29 + 10) + float(B) * A * (29 + 6)
    dyn_bytes = n_as * (C_ACT * 4 + 1 + 9 + 29 + 4) + float(B) * A * (29 + 6)      # k_rollout_dyn: action, mask, log x/y/valid in; sim row, log divergence out
    met_bytes = n_as * (21 + 6)                                                    # k_rollout_metrics: x, y, yaw, length, width, valid in; 2 flags + distance out
    fused_flops = pairs_eval * N_STEPS * FLOP_PER_PAIR
    roll_ms = dyn_ms + met_ms
    tr_dyn, src_dyn = profiled_traffic("k_rollout_dyn_bulk")          # A % 16 == 0: the bulk-staged variant runs
    if tr_dyn is None:
        tr_dyn, src_dyn = profiled_traffic("k_rollout_dyn")
    tr_met, src_met = profiled_traffic("k_rollout_metrics")
    roofline = {"bound": "hbm", "achieved": fused_bytes / (roll_ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                "frac": fused_bytes / (roll_ms * 1e-3) / 1e9 / hbm_peak,
                "traffic": (tr_dyn + tr_met) if (tr_dyn is not None and tr_met is not None) else None, "traffic_source": src_met,
                "kernel": "k_rollout_dyn_bulk + k_rollout_metrics (the rollout graph: one launch of each per 80-step rollout)",
                "kernel_ms": roll_ms, "graph_replay_ms": kf_ms, "algorithmic_bytes_per_launch": fused_bytes,
                "peak_source": hbm_src, "kernel_share_of_step": roll_ms / ms_step,
                "hbm_time_ms_at_peak": fused_bytes / (hbm_peak * 1e9) * 1e3,
                "kernels": {
                    "k_rollout_metrics": {"ms": met_ms, "share_of_step": met_ms / ms_step, "algorithmic_bytes_per_launch": met_bytes,
                                          "hbm_frac": met_bytes / (met_ms * 1e-3) / 1e9 / hbm_peak, "traffic": tr_met,
                                          "bound_observed": "instruction issue 77.5 % and LSU data-pipe wavefronts 71.5 % (ncu: profiles/r03_k_rollout_ncu.md), not HBM and not the FP32 pipe",
                                          "alu_frac_on_evaluated_pairs": fused_flops / (met_ms * 1e-3) / 1e12 / fp32_peak},
                    "k_rollout_dyn": {"ms": dyn_ms, "share_of_step": dyn_ms / ms_step, "algorithmic_bytes_per_launch": dyn_bytes,
                                      "hbm_frac": dyn_bytes / (dyn_ms * 1e-3) / 1e9 / hbm_peak, "traffic": tr_dyn}},
                "fp32_time_ms_at_peak_on_evaluated_pairs": fused_flops / (fp32_peak * 1e12) * 1e3,
                "pairs_bruteforce_per_step": pairs_per_launch, "pairs_evaluated_per_step": pairs_eval,
                "evaluated_fraction": pairs_eval / pairs_per_launch, "pairs_per_corner": ev_pairs / max(n_corner, 1),
                "slow_path_corner_fraction": n_slow / max(n_corner, 1),
                "alu_frac_bruteforce_equivalent": pairs_per_launch * N_STEPS * FLOP_PER_PAIR / (roll_ms * 1e-3) / 1e12 / fp32_peak,
                "note": "achieved = compulsory HBM bytes of the rollout / (k_rollout_dyn + k_rollout_metrics) CUDA-event time. The exact culling "
                        "(SURVEY 8(d)) leaves under 0.1 % of the corner-segment pairs, so the slower roof is the compulsory IO; the dominant "
                        "kernel k_rollout_metrics is bound by instruction issue (gathers through the cell lists), see DESIGN.md 7"}
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
                       "frac": bf_achieved / fp32_peak, "traffic": profiled_traffic("k_offroad")[0],
                       "kernel": "k_offroad (offroad_mode=WM_OFFROAD_BRUTE_FORCE)", "kernel_ms": kb_ms,
                       "pairs_per_launch": pairs_per_launch, "flop_per_pair": FLOP_PER_PAIR, "peak_source": peak_src,
                       "peak_measured": fp32_peak_measured, "frac_of_measured_peak": bf_achieved / fp32_peak_measured,
                       "peak_measured_source": "wm_selftest_ffma in this run: register-resident FFMA %.1f / FFMA2 %.1f TFLOP/s" % (fp32_measured["ffma"], fp32_measured["ffma2"])}
    clocks = sampler.stop() if rank == 0 else None
    others = None
    if rank == 0 and world == 1 and not args.no_extras:
        others, _ = other_configs(wm, ws, torch, hbm_peak, log_d, sim_d, stream)

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
        # parity on the same sample, teacher-forced (P16): the oracle's metrics on the GPU's OWN rows at 9 of the 80
        # steps, flags compared outside the 1e-4 m ambiguity band (P15), band members counted
        got = {k: v[:sb].cpu().numpy() for k, v in sim_d.items()}
        g_off = out_d["offroad"][:sb].cpu().numpy(); g_sd = out_d["offroad_dist"][:sb].cpu().numpy(); g_ov = out_d["overlap"][:sb].cpu().numpy()
        flags_equal, amb_corners, n_corners, amb_pairs, dist_ok, checked = True, 0, 0, 0, True, []
        for s_ in list(range(0, N_STEPS, 10)) + [N_STEPS - 1]:
            tt = cfg["t0"] + s_ + 1
            off = oracle.offroad(got, tt, rgs)
            v_ = got["valid"][:, tt] == 1
            amb = off["ambig"] == 1
            clean = v_ & ~amb.any(axis=1)
            flags_equal &= bool(np.array_equal(g_off[:, s_][clean], off["flag"][clean]))
            ref = off["signed_dist"].astype(np.float64)[clean]
            dist_ok &= bool(np.all(np.abs(g_sd[:, s_][clean].astype(np.float64) - ref) <= 1e-5 * np.abs(ref) + 3e-6))
            amb_corners += int((amb & v_[:, None, :]).sum()); n_corners += 4 * int(v_.sum())
            ovl = oracle.overlap(got, tt)
            band = np.abs(ovl["gap"]) < 1e-4
            cl = ~band.any(axis=2)
            flags_equal &= bool(np.array_equal(g_ov[:, s_][cl], ovl["flag"][cl]))
            amb_pairs += int(band.sum())
            checked.append(s_)
        cpu = {"value": sb * A * N_STEPS / dt, "unit": "agent-steps/s", "cores": oracle.num_threads(), "kind": "oracle",
               "sample": "first %d of %d scenarios x %d steps, oracle.rollout, %.1f s wall" % (sb, B, N_STEPS, dt),
               "offroad_flag_agreement_free_running": agree,
               "parity_teacher_forced": {"scenarios": sb, "steps_checked": checked, "flags_equal_outside_band": flags_equal,
                                         "distances_within_tolerance": dist_ok, "tolerance": "rel 1e-5 + 3e-6 m",
                                         "ambiguous_corners": amb_corners, "corners": n_corners, "ambiguous_overlap_pairs": amb_pairs}}

    if rank == 0:
        extra = {"prepare_ms": prepare_ms, "reset_ms": reset_ms, "value_incl_prepare": agent_steps / ((prepare_ms + ms_step) * 1e-3),
                 "grid_cells_without_list_frac": {k: v[2] for k, v in grid_stats.items()}}
        if roofline_bf:
            extra["bruteforce_frac"] = roofline_bf.get("frac")
        if others:
            o3, o5 = others["config3_observe"], others["config5_expert"]
            extra.update(ms_hist=o3["k_observe_hist"]["ms"], hist_hbm_frac=o3["k_observe_hist"]["hbm_frac"],
                         ms_topk=o3["k_observe_topk"]["ms"], topk_hbm_frac=o3["k_observe_topk"]["hbm_frac"],
                         ms_config2=others["config2_step"]["ms"], ms_config4=others["config4_stress"]["ms"],
                         config4_cells_without_list_frac=others["config4_stress"]["grid_cells_without_list_frac"],
                         ms_expert=o5["k_inverse_expert"]["ms"], ms_kinematic=o5["k_inverse_kinematic"]["ms"],
                         ms_vjp=o5["k_rollout_vjp"]["ms"], ms_idm_step=others["config5_idm"]["k_idm_step"]["ms"],
                         idm_workload=others["config5_idm"]["workload"])
        line = {
            "metric": METRIC, "value": value, "unit": "agent-steps/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": "config5: B=%d/GPU A=128 R=20000 T=91, 80-step InvertibleBicycle rollout + overlap + offroad + log divergence, one CUDA graph" % B,
                       "B_per_gpu": B, "A": A, "R": R, "T": T, "n_steps": N_STEPS, "S_e_max": int(seg_max),
                       "S_e_mean": float(n_seg.mean()), "l2": "inputs exceed L2 (segments %.2f GB + state per step)" % (n_seg.sum() * 24 / 1e9),
                       "parallelism": "scenario shards, no collective", "valid_agent_steps_per_s": valid_value,
                       "ms_per_sim_step": ms_step / N_STEPS,
                       "value_counts": "agent SLOTS (valid or not, SURVEY 8(d)); valid_agent_steps_per_s counts the valid ones",
                       **extra},
            # wm_prepare = the static precompute a NEW batch of scenarios needs before its first rollout (outside `value`:
            # `value` assumes prepared scenarios, e.g. re-rolled in training); value_incl_prepare = one prepare per rollout
            "prepare_ms": prepare_ms, "reset_ms": reset_ms,
            "value_incl_prepare": agent_steps / ((prepare_ms + ms_step) * 1e-3),
            "other_configs": others,
            "roofline": roofline, "roofline_offroad_grid": roofline_grid, "roofline_bruteforce": roofline_bf, "step_roofline": step_roofline,
            "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
        }
        print(json.dumps(line))
    wm.wm_destroy(h)
    return 0


if __name__ == "__main__":
    sys.exit(main())
