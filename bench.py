#!/usr/bin/env python
"""bench.py — PSDF value+grad throughput on the BASELINE workload (contract in the task brief).

A "step" is one pass of the whole hot path (H1-H8: pose setup, both pools, SAT, min over
obstacles, witness gradient) over one batch of synthetic poses, i.e. ONE psdf_eval call.
Default workload: config 5 (throughput stress, the largest single-GPU config, the one
BASELINE.json's ">= 60 % of the FP32 roofline" is quoted on).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 3|4|5] [--impl reference]

Prints ONE JSON line on rank 0.  `--impl reference` times the CPU oracle as it stands on
the host cores on a bounded sample of the same workload (no GPU work).
"""
from __future__ import annotations

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

METRIC = "psdf_value_grad_pose_obstacle_pairs_per_s"
UNIT = "pairs/s"
FP32_LANES_PER_SM = 128            # B200 SM: 4 SMSPs x 32 FP32 lanes (guide: blackwell_cuda_programming.md)


def flops_per_launch(w) -> float:
    """Algorithmic FLOPs, fixed before tuning:
    F(V,e) = 32 V e + 6 e + 4 V + 6 per (pose, obstacle with e valid edges)."""
    e = w.valid_edges().astype(np.float64)
    e = e[e > 0]
    V = w.V
    return float(w.N) * float((32.0 * V * e + 6.0 * e + 4.0 * V + 6.0).sum())


def algorithmic_bytes(w) -> float:
    return w.N * (12 + 16) + int(w.valid_edges().sum()) * 32.0


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            self.t = threading.Thread(target=lambda: self.lines.extend(self.proc.stdout), daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.t.join(timeout=2)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for k, nm in enumerate(names):
                if f[3 + k].lower() == "active":
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def load_workload(idx: int, rank: int):
    from paper_2607_04310_b200 import workloads as W
    w = W.make_config(idx)
    if rank > 0:                       # weak scaling: same scene, a different pose batch per rank
        w.poses = w.poses.copy()
        w.poses[:, 2] += np.float32(0.37 * rank)
    return w


def measured_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except (OSError, ValueError):
        return {}


def ncu_traffic(workload_name: str, column: int = 1):
    """Per-launch DRAM bytes (column 1) or executed warp instructions (column 2) of the dominant
    kernel from the committed ncu --set full capture (profiles/traffic.csv), or None."""
    try:
        for ln in open(os.path.join(ROOT, "profiles", "traffic.csv")).read().splitlines()[1:]:
            f = ln.split(",")
            if f[0] == workload_name:
                return float(f[column])
    except (OSError, ValueError, IndexError):
        pass
    return None


def _pct(xs_us):
    a = np.sort(np.asarray(xs_us))
    return {"p50_us": float(a[len(a) // 2]), "p95_us": float(a[int(len(a) * 0.95)]),
            "p99_us": float(a[int(len(a) * 0.99)]), "min_us": float(a[0]), "n": int(len(a))}


def mpc_latency(torch, psdf, replays=2000):
    """p50/p95/p99 end-to-end latency of the MPC-sized configs (BASELINE.json configs[0], [1]):
    psdf_eval_host = host poses -> pinned staging -> CUDA-graph {H2D, kernel, D2H} -> host results,
    timed on the host clock around the C-ABI call; kernel-only by CUDA events around psdf_eval.
    Also the paper's Table-I shape sweep (context, other hardware)."""
    from paper_2607_04310_b200 import workloads as W
    out = {}

    def host_lat(scene, w, n_rep, grad=True, per_obs=False, coeffs=False, bound=True):
        value = np.empty(w.N, np.float32)
        g = np.empty((w.N, 3), np.float32) if grad else None
        po = np.empty((w.N, w.M), np.float32) if per_obs else None
        if coeffs:       # pre-marshalled calls (Scene.bind_*): what an MPC loop with fixed buffers makes
            call = scene.bind_mpc_coeffs_host(w.poses, np.empty((w.N, 4), np.float32), 0.3, 0.05, 0.05)
        elif bound:
            call = scene.bind_eval_host(w.poses, value, g, po)
        else:            # marshalling on every call (numpy pointer extraction: ~2 us per array)
            call = lambda: scene.eval_host_into(w.poses, value, g, po)
        for _ in range(500):        # ~10 ms: the first calls of a process run ~5 us slower
            call()
        ts = []
        for _ in range(n_rep):
            t0 = time.perf_counter_ns()
            call()
            ts.append((time.perf_counter_ns() - t0) * 1e-3)
        return _pct(ts)

    def kernel_lat(scene, w, n_rep=300, per_obs=False):
        poses = torch.from_numpy(w.poses).cuda()
        value = torch.empty(w.N, dtype=torch.float32, device="cuda")
        grad = torch.empty((w.N, 3), dtype=torch.float32, device="cuda")
        po = torch.empty((w.N, w.M), dtype=torch.float32, device="cuda") if per_obs else False
        st = torch.cuda.current_stream()
        for _ in range(20):
            scene.eval(poses, value=value, grad=grad, per_obstacle=po, stream=st)
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_rep)]
        for a, b in evs:
            a.record(st)
            scene.eval(poses, value=value, grad=grad, per_obstacle=po, stream=st)
            b.record(st)
        torch.cuda.synchronize()
        return _pct([a.elapsed_time(b) * 1e3 for a, b in evs])

    for idx in (1, 2):
        w = W.make_config(idx)
        scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=w.N)
        e = {"N": w.N, "M": w.M, "pairs": w.n_pairs(),
             "eval_host_value_grad": host_lat(scene, w, replays),
             "kernel_only_value_grad": kernel_lat(scene, w)}
        if idx == 1:
            e["eval_host_value_grad_marshalled_per_call"] = host_lat(scene, w, replays, bound=False)
            e["mpc_coeffs_host"] = host_lat(scene, w, replays, coeffs=True)
        else:
            e["eval_host_value_grad_per_obstacle"] = host_lat(scene, w, replays, per_obs=True)
        out[w.name] = e
        scene.close()
    t1 = {}
    for M in (1, 10, 100):
        for B in (1, 15, 100):
            w = W.table1_case(M, B)
            scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=w.N)
            t1[f"M{M}_B{B}"] = host_lat(scene, w, 500)["p50_us"]
            scene.close()
    out["table1_shapes_eval_host_p50_us"] = t1
    out["table1_paper_rtx4090_ms"] = {"M1_B1": 1.981, "M1_B15": 2.154, "M1_B100": 2.212, "M10_B1": 2.152,
                                      "M10_B15": 2.213, "M10_B100": 2.250, "M100_B1": 2.221, "M100_B15": 2.222,
                                      "M100_B100": 2.207,
                                      "note": "PAPER.md:417-419 Table I, PSDF rows (PyTorch graph incl. backward, "
                                              "RTX 4090): context only, other hardware"}
    out["clock"] = ("host perf_counter_ns around the Python binding's pre-marshalled C-ABI call (Scene.bind_eval_host / "
                    "bind_mpc_coeffs_host: the ctypes foreign call is inside, numpy pointer extraction is done once)")
    return out


def run_reference(args, w):
    """--impl reference: the oracle, as it stands, on the host cores; each step is a bounded
    sample (`--ref-poses` poses of the workload, value+grad)."""
    from oracle import psdf_oracle as O
    # bounded sample: calibrate on 64 poses, then size the per-step sample so that the whole
    # --steps/--warmup run takes about --ref-seconds on this box's cores
    cal = w.subsample(min(64, w.N))
    t0 = time.perf_counter()
    O.evaluate(cal.footprint, cal.A, cal.B, cal.S, cal.poses)
    rate = cal.N / max(time.perf_counter() - t0, 1e-6)                       # poses/s
    n = int(min(args.ref_poses, w.N, max(32, rate * args.ref_seconds / (args.steps + min(args.warmup, 1)))))
    sub = w.subsample(n)
    for _ in range(min(args.warmup, 1)):
        O.evaluate(sub.footprint, sub.A, sub.B, sub.S, sub.poses)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        O.evaluate(sub.footprint, sub.A, sub.B, sub.S, sub.poses)
    dt = (time.perf_counter() - t0) / args.steps
    val = sub.n_pairs() / dt
    cores = O.max_threads()
    sample = f"{n} of {w.N} poses (stride subsample) x {w.M} obstacles per step, value+grad, float64"
    return {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{w.name} (BASELINE.json configs[{args.workload - 1}]), value+grad", "N": n, "M": w.M, "E": w.E, "V": w.V, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--workload", type=int, default=5, choices=[3, 4, 5])
    ap.add_argument("--impl", default="psdf", choices=["psdf", "reference"])
    ap.add_argument("--ref-poses", type=int, default=4096)
    ap.add_argument("--ref-seconds", type=float, default=90.0, help="--impl reference: target total run time")
    ap.add_argument("--cpu-poses", type=int, default=16384, help="upper limit of the cpu_baseline pose sample")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target oracle time of the cpu_baseline sample")
    ap.add_argument("--no-latency", action="store_true", help="skip the MPC-sized latency section")
    ap.add_argument("--value-only", action="store_true", help="extra run without gradients is always reported; "
                    "this flag makes it the headline")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        if rank == 0:
            print(json.dumps(run_reference(args, load_workload(args.workload, 0))), flush=True)
        return 0

    import torch
    import torch.distributed as dist
    from paper_2607_04310_b200 import psdf, sharding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    w = load_workload(args.workload, rank)
    scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=w.N)
    poses = torch.from_numpy(w.poses).cuda()
    value = torch.empty(w.N, dtype=torch.float32, device="cuda")
    grad = torch.empty((w.N, 3), dtype=torch.float32, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2
    stream = torch.cuda.current_stream()

    def timed(n_steps, with_grad):
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_steps)]
        for a, b in evs:
            flush.zero_()                                    # L2 flush between timed iterations
            a.record(stream)
            scene.eval(poses, value=value, grad=grad if with_grad else False, stream=stream)
            b.record(stream)
        torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in evs]

    timed(max(args.warmup, 3), True)
    fp32_meas = psdf.psdf_measure_fp32_peak(8192) if rank == 0 else None
    timed(3, True)
    sampler = ClockSampler(local_rank)
    n_launch0 = psdf.psdf_kernel_launches()
    barrier()
    sampler.start()
    t_wall0 = time.perf_counter()
    times = timed(args.steps, not args.value_only)
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    launches = psdf.psdf_kernel_launches() - n_launch0
    t_dev = float(np.sum(times)) * 1e-3
    other = timed(max(args.steps // 4, 5), args.value_only)     # the other variant, for the record

    # exact broad-phase culling (psdf_set_culling): same outputs, bit for bit
    scene.set_culling(True)
    timed(5, True)
    scene.cull_stats()
    k_cull = max(args.steps // 2, 10)
    cull_times = timed(k_cull, True)
    eval_pairs, edge_steps = scene.cull_stats()
    v_cull = value.clone()
    scene.set_culling(False)
    timed(1, True)
    culled_same = bool(torch.equal(v_cull, value))

    # end to end through the public host API: pinned staging + H2D + kernel + D2H inside
    for _ in range(3):
        scene.eval_host(w.poses, grad=True)
    barrier()
    k_e2e = max(args.steps // 4, 5)
    t0 = time.perf_counter()
    for _ in range(k_e2e):
        scene.eval_host(w.poses, grad=True)
    t_e2e = (time.perf_counter() - t0) / k_e2e

    t_dev, t_e2e, t_wall = sharding.max_over_ranks([t_dev, t_e2e, t_wall])      # max over ranks

    if rank == 0:
        pairs = w.n_pairs()
        F = flops_per_launch(w)
        t_kernel = float(np.mean(times)) * 1e-3              # average launch duration, CUDA events
        peaks = measured_peaks()
        sm_max = float(peaks.get("sm_max_mhz", 1965.0))
        sms = torch.cuda.get_device_properties(0).multi_processor_count
        peak_nominal = sms * FP32_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
        achieved = F / t_kernel / 1e12
        hbm = float(peaks.get("hbm_gbs", 6650.0))
        # SURVEY.md 8(d) issue-slot view: executed lane-instructions/s against one instruction per
        # lane and clock (= P_fp32 / 2); the instruction count is the committed ncu capture's.
        warp_inst = ncu_traffic(w.name, 2)
        issue_view = None
        if warp_inst:
            issue_peak = sms * FP32_LANES_PER_SM * sm_max * 1e6
            issue_view = {"warp_inst_per_launch": warp_inst, "lane_inst_per_s": warp_inst * 32 / t_kernel,
                          "peak_lane_inst_per_s": issue_peak, "frac": warp_inst * 32 / t_kernel / issue_peak,
                          "source": "smsp__inst_executed.sum of the committed ncu --set full capture (profiles/traffic.csv)"}
        out = {
            "metric": METRIC, "value": pairs * world * args.steps / t_dev, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": t_dev / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"{w.name} (BASELINE.json configs[{args.workload - 1}]), "
                                   f"{'value-only' if args.value_only else 'value+grad'}",
                       "N_per_gpu": w.N, "M": w.M, "E": w.E, "V": w.V, "pairs_per_gpu": pairs,
                       "valid_edges": int(w.valid_edges().sum()), "l2_flush": "256 MiB memset between timed launches",
                       "parallelism": f"replicated scene, pose-sharded x{world}", "seed": 43100 + args.workload},
            "roofline": {"bound": "alu", "achieved": achieved, "peak": peak_nominal, "unit": "TFLOP/s",
                         "frac": achieved / peak_nominal, "traffic": ncu_traffic(w.name),
                         "peak_source": f"derived: {sms} SMs x {FP32_LANES_PER_SM} FP32 lanes x 2 x {sm_max:.0f} MHz "
                                        "(clocks.max.sm, MEASURED_PEAKS.json); no FP32 figure in MEASURED_PEAKS.json",
                         "flops_per_launch": F, "flop_formula": "32*V*e+6*e+4*V+6 per (pose, obstacle), valid edges only",
                         "kernel_ms": t_kernel * 1e3, "kernel_ms_min": float(np.min(times)),
                         "kernel_ms_median": float(np.median(times)), "issue_slot_view": issue_view,
                         "peak_measured_ffma": fp32_meas, "frac_of_measured_ffma": achieved / fp32_meas if fp32_meas else None,
                         "hbm_bytes_algorithmic": algorithmic_bytes(w),
                         "hbm_gbs_achieved": algorithmic_bytes(w) / t_kernel / 1e9, "hbm_gbs_peak_measured": hbm},
            "other_variant": {"what": "value+grad" if args.value_only else "value-only",
                              "ms_per_step": float(np.mean(other)), "value": pairs / (float(np.mean(other)) * 1e-3)},
            "e2e": {"value": pairs * world / t_e2e, "unit": UNIT, "ms_per_step": t_e2e * 1e3,
                    "h2d_bytes_per_step": w.N * 12, "d2h_bytes_per_step": w.N * 16,
                    "api": "psdf_eval_host (host buffers -> pinned staging -> CUDA graph {H2D, kernel, D2H} -> host)"},
            "culling": {"what": "psdf_set_culling(1): obstacle grid + bounding-circle / oriented-box lower bounds, "
                                "pair-queue kernel, value+grad; outputs bit-identical to the dense path "
                                "(checked in this run: %s)" % culled_same,
                        "ms_per_step": float(np.mean(cull_times)), "value": pairs / (float(np.mean(cull_times)) * 1e-3),
                        "unit": UNIT, "speedup_vs_dense": t_kernel * 1e3 / float(np.mean(cull_times)),
                        "evaluated_pair_fraction": eval_pairs / k_cull / pairs,
                        "evaluated_flops_per_step": ((32.0 * w.V + 6.0) * edge_steps + (4.0 * w.V + 6.0) * eval_pairs) / k_cull,
                        "note": "pairs/s counts all pairs (SURVEY.md 8(d)); culled pairs cost at most two bound tests"},
            "gpu_launches": int(launches), "wall_s_timed_region": t_wall, "clocks": clocks,
            "paper_context": {"psdf_rtx4090_M100_B100_ms": 2.207, "implied_pairs_per_s": 4.5e6,
                              "source": "PAPER.md:419 Table I (other hardware, context only)"},
        }
        if world == 1:
            from oracle import psdf_oracle as O          # cpu_baseline leg: the oracle as it stands
            cal = w.subsample(min(256, w.N))             # size the sample for ~cpu_seconds on THIS host
            t0 = time.perf_counter()
            O.evaluate(cal.footprint, cal.A, cal.B, cal.S, cal.poses)
            rate = cal.N / (time.perf_counter() - t0)
            sub = w.subsample(int(min(max(args.cpu_seconds * rate, 1024), args.cpu_poses, w.N)))
            t0 = time.perf_counter()
            O.evaluate(sub.footprint, sub.A, sub.B, sub.S, sub.poses)
            dt = time.perf_counter() - t0
            out["cpu_baseline"] = {"value": sub.n_pairs() / dt, "unit": UNIT, "cores": O.max_threads(),
                                   "kind": "oracle", "seconds": dt,
                                   "sample": f"{sub.N} of {w.N} poses (stride subsample) x {w.M} obstacles, "
                                             "value+grad, float64, OpenMP"}
            one = w.subsample(int(min(max(0.25 * args.cpu_seconds * rate / max(O.max_threads(), 1), 64), w.N)))
            t0 = time.perf_counter()
            O.evaluate(one.footprint, one.A, one.B, one.S, one.poses, nthreads=1)
            dt1 = time.perf_counter() - t0
            out["cpu_baseline"]["single_thread"] = {"value": one.n_pairs() / dt1, "unit": UNIT, "seconds": dt1,
                                                    "sample": f"{one.N} of {w.N} poses (stride subsample), 1 thread"}
            if not args.no_latency:
                out["mpc_latency"] = mpc_latency(torch, psdf)
        print(json.dumps(out), flush=True)
    scene.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
