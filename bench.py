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
                                          "-lms", "25", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
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
    kernel from the committed ncu --set full capture (profiles/traffic.csv), or None; column 3 is the
    commit whose code was captured (a string)."""
    try:
        for ln in open(os.path.join(ROOT, "profiles", "traffic.csv")).read().splitlines()[1:]:
            f = ln.split(",")
            if f[0] == workload_name:
                return f[column] if column == 3 else float(f[column])
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
        out = _pct(ts)
        # the same call timed INSIDE the library (steady_clock around the C-ABI entry point: no
        # interpreter, no ctypes in the timed region)
        inlib = scene.bench_host_latency(w.poses, n_rep, grad=grad, per_obstacle=per_obs,
                                         coeffs=(0.3, 0.05, 0.05) if coeffs else None)
        out["c_abi_clock"] = _pct(inlib)
        return out

    def serve_lat(scene, w, n_rep, coeffs=None):
        """psdf_serve_step (persistent kernel + mapped-memory mailbox): same clocks as host_lat."""
        scene.serve_begin(w.N, coeffs=coeffs, idle_timeout_ms=200)
        rows = np.empty((w.N, 4), np.float32)
        call = scene.bind_serve_step(w.poses, rows)
        for _ in range(500):
            call()
        ts = []
        for _ in range(n_rep):
            t0 = time.perf_counter_ns()
            call()
            ts.append((time.perf_counter_ns() - t0) * 1e-3)
        out = _pct(ts)
        out["c_abi_clock"] = _pct(scene.bench_serve_latency(w.poses, n_rep))
        scene.serve_end()
        return out

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
            e["serve_step_mpc_coeffs"] = serve_lat(scene, w, replays, coeffs=(0.3, 0.05, 0.05))
        else:
            e["eval_host_value_grad_per_obstacle"] = host_lat(scene, w, replays, per_obs=True)
        e["serve_step_value_grad"] = serve_lat(scene, w, replays)
        out[w.name] = e
        scene.close()
    t1, t1s = {}, {}
    for M in (1, 10, 100):
        for B in (1, 15, 100):
            w = W.table1_case(M, B)
            scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=w.N)
            t1[f"M{M}_B{B}"] = host_lat(scene, w, 500)["p50_us"]
            t1s[f"M{M}_B{B}"] = serve_lat(scene, w, 500)["p50_us"]
            scene.close()
    out["table1_shapes_eval_host_p50_us"] = t1
    out["table1_shapes_serve_step_p50_us"] = t1s
    out["serve_step"] = ("psdf_serve_begin / psdf_serve_step: persistent lane-split kernel polling a mailbox in pinned, "
                         "device-mapped memory; no launch and no stream synchronisation per control cycle; rows "
                         "bit-identical to psdf_eval_host / psdf_mpc_coeffs_host (tests/test_gpu_serve.py)")
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


def pinned(torch, shape):
    """Page-locked host array (numpy view of a pinned torch tensor): what a caller that cares about
    end-to-end time hands to psdf_eval_host (include/psdf.h: pinned buffers are used in place)."""
    return torch.empty(shape, dtype=torch.float32, pin_memory=True).numpy()


class DeviceRun:
    """One workload resident in HBM: scene, poses, outputs, and the timed psdf_eval loop."""

    def __init__(self, torch, psdf, w, flush):
        self.torch, self.w, self.flush = torch, w, flush
        self.scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=w.N)
        self.poses = torch.from_numpy(w.poses).cuda()
        self.value = torch.empty(w.N, dtype=torch.float32, device="cuda")
        self.grad = torch.empty((w.N, 3), dtype=torch.float32, device="cuda")
        self.stream = torch.cuda.current_stream()

    def timed(self, n_steps, with_grad=True):
        """n_steps psdf_eval calls, L2 flushed before each, CUDA events on the launching stream."""
        torch = self.torch
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_steps)]
        for a, b in evs:
            self.flush.zero_()                               # L2 flush between timed iterations
            a.record(self.stream)
            self.scene.eval(self.poses, value=self.value, grad=self.grad if with_grad else False, stream=self.stream)
            b.record(self.stream)
        torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in evs]

    def timed_trajectories(self, n_steps, T, H, d_safe=0.5):
        """As `timed`, for psdf_eval_trajectories (evaluation + per-trajectory reductions, one launch)."""
        torch = self.torch
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_steps)]
        for a, b in evs:
            self.flush.zero_()
            a.record(self.stream)
            self.scene.eval_trajectories(self.poses, T, H, d_safe, grad=True, stream=self.stream)
            b.record(self.stream)
        torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in evs]

    def e2e(self, n_steps, pin):
        """n_steps psdf_eval_host calls from HOST buffers (host clock; H2D and D2H inside).  Returns
        (seconds per step, value, grad) with the outputs of the last call."""
        w = self.w
        if pin:
            p, v, g = pinned(self.torch, (w.N, 3)), pinned(self.torch, (w.N,)), pinned(self.torch, (w.N, 3))
            p[:] = w.poses
        else:
            p, v, g = w.poses, np.empty(w.N, np.float32), np.empty((w.N, 3), np.float32)
        for _ in range(3):
            self.scene.eval_host_into(p, v, g)
        v[:] = 0
        g[:] = 0
        t0 = time.perf_counter()
        for _ in range(n_steps):
            self.scene.eval_host_into(p, v, g)
        return (time.perf_counter() - t0) / n_steps, v, g


def parity_report(torch, psdf, O, workloads, budget_poses):
    """BASELINE.md section 3 / SURVEY.md 5: GPU against the oracle on all five configs, measured exactly
    as tests/parity.py does (|d value|, gradient relative error where the oracle's arg-min margin
    allows, compared and penetrating fractions).  Configs 1-2 whole, 3-5 on a random sample of the
    FULL-size launch's outputs.  Runs outside every timed region; the oracle calls here belong to
    the cpu_baseline leg (the same oracle, the same host cores)."""
    from tests.parity import stats, VALUE_TOL, GRAD_REL_TOL
    out = {"bar": {"value_tol_m": VALUE_TOL, "grad_rel_tol": GRAD_REL_TOL, "margin_min_m": 1e-4,
                   "rule": "gradient compared where the oracle's arg-min margin > 1e-4 m; on the separated branch also "
                           "phi > 1e-3 m (DESIGN.md reading G9)"}}
    for idx, w in workloads.items():
        scene = psdf.Scene(w.footprint, w.A, w.B, w.S, max_poses=w.N)
        v, g, po = scene.eval(torch.from_numpy(w.poses).cuda(), grad=True, per_obstacle=(idx == 2))
        torch.cuda.synchronize()
        v, g = v.cpu().numpy(), g.cpu().numpy()
        n = min(w.N, budget_poses[idx])
        sel = np.sort(np.random.default_rng(777 + idx).choice(w.N, n, replace=False))
        ref = O.evaluate(w.footprint, w.A, w.B, w.S, w.poses[sel], per_obstacle=(idx == 2))
        st = stats(ref, v[sel], g[sel], po.cpu().numpy()[sel] if idx == 2 else None)
        st = {k: st[k] for k in st if not k.startswith("argmax")}
        st["sample"] = f"{n} of {w.N} poses of the full-size launch" if n < w.N else f"all {w.N} poses"
        st["within_bar"] = bool(st["inf_pattern_equal"] and st["max_dvalue"] <= VALUE_TOL and st["max_grad_rel"] <= GRAD_REL_TOL)
        out[w.name] = st
        scene.close()
    return out


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
    ap.add_argument("--no-extras", action="store_true", help="skip per_config, parity and latency (profiling runs)")
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
    if os.environ.get("PSDF_BENCH_SHUFFLE"):                  # diagnostic: destroys the spatial coherence of trajectory batches
        w.poses = w.poses[np.random.default_rng(1).permutation(w.N)].copy()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2
    run = DeviceRun(torch, psdf, w, flush)
    scene, value, grad = run.scene, run.value, run.grad

    run.timed(max(args.warmup, 3), True)
    fp32_meas = psdf.psdf_measure_fp32_peak(8192) if rank == 0 else None
    run.timed(3, True)
    sampler = ClockSampler(local_rank)
    n_launch0 = psdf.psdf_kernel_launches()
    barrier()
    sampler.start()
    t_wall0 = time.perf_counter()
    times = run.timed(args.steps, not args.value_only)
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    launches = psdf.psdf_kernel_launches() - n_launch0
    t_dev = float(np.sum(times)) * 1e-3
    other = run.timed(max(args.steps // 4, 5), args.value_only)     # the other variant, for the record
    run.timed(1, True)
    v_dense, g_dense = value.cpu().numpy(), grad.cpu().numpy()

    # exact broad-phase culling (psdf_set_culling): same outputs, bit for bit
    scene.set_culling(True)
    run.timed(5, True)
    scene.cull_stats()
    k_cull = max(args.steps // 2, 10)
    cull_times = run.timed(k_cull, True)
    eval_pairs, edge_steps = scene.cull_stats()
    culled_same = bool(np.array_equal(value.cpu().numpy(), v_dense) and np.array_equal(grad.cpu().numpy(), g_dense))
    # ... and end to end through psdf_eval_host, from pinned and from ordinary host buffers
    k_e2e = max(args.steps // 4, 5)
    t_e2e_cull, vc, gc = run.e2e(4 * k_e2e, pin=True)
    e2e_cull_checked = bool(np.array_equal(vc, v_dense) and np.array_equal(gc, g_dense))
    t_e2e_cull_pageable, _, _ = run.e2e(k_e2e, pin=False)
    scene.set_culling(False)

    # end to end through the public host API (dense): H2D + kernels + D2H inside the timed region
    barrier()
    t_e2e, ve, ge = run.e2e(k_e2e, pin=True)
    e2e_checked = bool(np.array_equal(ve, v_dense) and np.array_equal(ge, g_dense))   # outside the timed region
    t_e2e_pageable, vp_, gp_ = run.e2e(k_e2e, pin=False)
    e2e_checked = e2e_checked and bool(np.array_equal(vp_, v_dense) and np.array_equal(gp_, g_dense))

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
                         "traffic_source": "profiles/traffic.csv: one ncu --set full capture of this kernel, code of commit "
                                           f"{ncu_traffic(w.name, 3)} (a constant of that capture, not of this run)",
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
                    "api": "psdf_eval_host from pinned host buffers (used in place): captured CUDA graph of "
                           "{H2D pose chunk, kernel, D2H result chunk} branches, stream synchronise",
                    "from_pageable_buffers_ms_per_step": t_e2e_pageable * 1e3},
            "e2e_outputs_checked": e2e_checked,
            "culling": {"what": "psdf_set_culling(1): obstacle grid + bounding-circle / oriented-box lower bounds, "
                                "pair-queue kernel, value+grad; outputs bit-identical to the dense path "
                                "(checked in this run: %s)" % culled_same,
                        "ms_per_step": float(np.mean(cull_times)), "value": pairs / (float(np.mean(cull_times)) * 1e-3),
                        "unit": UNIT, "speedup_vs_dense": t_kernel * 1e3 / float(np.mean(cull_times)),
                        "evaluated_pair_fraction": eval_pairs / k_cull / pairs,
                        "evaluated_flops_per_step": ((32.0 * w.V + 6.0) * edge_steps + (4.0 * w.V + 6.0) * eval_pairs) / k_cull,
                        "e2e_culled": {"ms_per_step": t_e2e_cull * 1e3, "value": pairs / t_e2e_cull, "unit": UNIT,
                                       "over_kernel": t_e2e_cull * 1e3 / float(np.mean(cull_times)),
                                       "outputs_checked": e2e_cull_checked,
                                       "from_pageable_buffers_ms_per_step": t_e2e_cull_pageable * 1e3,
                                       "api": "psdf_eval_host with culling on, pinned host buffers (one launch reading and writing them over PCIe)"},
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
            if not args.no_extras:
                from paper_2607_04310_b200 import workloads as W
                allw = {i: (w if i == args.workload else W.make_config(i)) for i in (1, 2, 3, 4, 5)}
                # roofline fraction of the other large configs (value+grad), same protocol as the headline
                per = {}
                for i in (3, 4, 5):
                    r = run if i == args.workload else DeviceRun(torch, psdf, allw[i], flush)
                    if i == args.workload:
                        tk = t_kernel
                    else:
                        r.timed(5)
                        tk = float(np.mean(r.timed(max(args.steps // 2, 10)))) * 1e-3
                    Fi = flops_per_launch(allw[i])
                    per[allw[i].name] = {"ms_per_step": tk * 1e3, "pairs_per_s": allw[i].n_pairs() / tk,
                                         "tflops": Fi / tk / 1e12, "frac": Fi / tk / 1e12 / peak_nominal,
                                         "N": allw[i].N, "M": allw[i].M, "V": allw[i].V, "what": "value+grad, dense"}
                    tr = allw[i].meta.get("n_traj")
                    if tr:          # trajectory batches: the same launch with the per-trajectory reductions fused in
                        Hs = allw[i].N // tr
                        r.timed_trajectories(3, tr, Hs)
                        tt = float(np.mean(r.timed_trajectories(max(args.steps // 2, 10), tr, Hs)))
                        per[allw[i].name]["with_fused_trajectory_reductions_ms"] = tt
                        per[allw[i].name]["fused_over_plain"] = tt / (tk * 1e3)
                    if i == 3:      # per-pose obstacle row windows (psdf_eval_windows, lane-split kernel at any N) at this size
                        wi = allw[i]
                        stage = np.arange(wi.N, dtype=np.int64) % 50
                        w0 = (stage * (wi.M - 64) // 49).astype(np.int32)            # a 64-row window sliding with the stage
                        win = torch.from_numpy(np.stack([w0, w0 + 64], 1).astype(np.int32)).cuda()
                        full = torch.from_numpy(np.tile(np.array([[0, wi.M]], np.int32), (wi.N, 1))).cuda()
                        for name, wt in (("eval_windows_64_rows_ms", win), ("eval_windows_all_rows_ms", full)):
                            for _ in range(3):
                                r.scene.eval_windows(r.poses, wt, grad=True)
                            evs = []
                            for _ in range(10):
                                flush.zero_()
                                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                                a.record(r.stream)
                                r.scene.eval_windows(r.poses, wt, grad=True, stream=r.stream)
                                b.record(r.stream)
                                evs.append((a, b))
                            torch.cuda.synchronize()
                            per[wi.name][name] = float(np.mean([a.elapsed_time(b) for a, b in evs]))
                    if i != args.workload:
                        r.scene.close()
                out["per_config"] = per
                out["parity"] = parity_report(torch, psdf, O, allw, {1: 20, 2: 50, 3: 3000, 4: 1200, 5: 1000})
                if not args.no_latency:
                    out["mpc_latency"] = mpc_latency(torch, psdf)
        print(json.dumps(out), flush=True)
    scene.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
