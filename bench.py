#!/usr/bin/env python
"""bench.py -- throughput of the stroke-expansion hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c4|c5|c3] [--impl ours|reference]

A step is one pass of the whole hot path (tag scan -> count -> allocation scan -> write) over one synthetic scene
(default: config 4, the CAD-scale scene BASELINE.json's target is quoted on: 1,000,000 segments, arc output,
tolerance 0.1).  `value` is input segments per second with the streams resident in HBM, device-timed with CUDA
events on the launching stream (L2 flushed between steps); `e2e` is the same metric through the host-buffer C-ABI
call with the H2D / D2H copies inside the timed region.  `--impl reference` times the CPU oracle instead.
Prints ONE JSON line (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "input path segments/sec expanded (device-timed)"
UNIT = "segments/s"
MODE_OF = {"c3": 0, "c4": 1, "c5": 0, "c1": 0, "c2": 0}
# dram__bytes_read.sum + dram__bytes_write.sum of the write pass per launch, from the committed ncu captures
# (profiles/r1_final.md); None = not captured for that workload
NCU_TRAFFIC = {"c4": 519.2e6, "c5": None}  # c4: 362.7 MB k_write_pieces + 156.5 MB k_write_segments (profiles/r1_final.md)
REF_SAMPLE_PATHS = {"c4": 20000, "c5": 1000, "c3": 20000, "c1": 256, "c2": 2000}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz, self._stop_evt = index, [], set(), None, threading.Event()

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = int(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
            names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                     "hw_power_brake_slowdown": 0x80, "sync_boost": 0x10, "applications_clocks_setting": 0x2}
            while not self._stop_evt.is_set():
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
                time.sleep(0.002)
        except Exception as e:  # no NVML: report that, never fake numbers
            self.reasons.add(f"nvml_unavailable:{type(e).__name__}")

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        med = int(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def max_over_ranks(seconds, world, device=None):
    """Device-timed seconds of this rank -> the maximum over all ranks (identity at world 1)."""
    if world <= 1:
        return float(seconds)
    import torch
    import torch.distributed as dist
    tt = torch.tensor([seconds], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return float(tt.item())


def job_throughput(units_per_rank_per_step, steps, world, seconds_max):
    """Whole-job throughput of `world` replicas (weak scaling): all ranks' units over the slowest rank's time."""
    return world * units_per_rank_per_step * steps / seconds_max


def make_scene(workload, n_paths=None):
    from paper_2405_00127_b200 import scenes as S
    return S.make(workload, n_paths=n_paths)


def time_oracle(sc, mode, reps=1):
    import oracle
    best, r = None, None
    for _ in range(reps):
        t0 = time.perf_counter()
        r = oracle.expand(sc.tags, sc.points, sc.styles, sc.affine, sc.tolerance, mode)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return best, r


def run_reference(args):
    """The oracle, as it stands, on the host cores (single thread), each step a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    mode = MODE_OF[args.workload] if args.mode is None else int(args.mode == "arc")
    npaths = REF_SAMPLE_PATHS[args.workload]
    sc = make_scene(args.workload, n_paths=npaths)
    for _ in range(args.warmup):
        time_oracle(sc, mode)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _, r = time_oracle(sc, mode)
    dt = time.perf_counter() - t0
    value = sc.n_segments * args.steps / dt
    sample = f"first {npaths} paths of {args.workload} ({sc.n_segments} segments -> {r.n_rec} records) per step"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": args.workload, "mode": "arc" if mode else "line", "tolerance": float(sc.tolerance), "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2405_00127_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    mode = MODE_OF[args.workload] if args.mode is None else int(args.mode == "arc")
    sc = make_scene(args.workload, n_paths=args.paths)  # replicas only: every rank expands the whole scene
    n_seg, n_paths = sc.n_segments, sc.n_paths
    tags, pts, sty = B.scene_to_torch(sc, device=dev)
    width = 8 if mode else 4
    ctx = B.sx_create(local)
    stream = torch.cuda.current_stream()
    poff = torch.empty(n_paths + 1, dtype=torch.int64, device=dev)
    total = B.sx_count(ctx, tags, pts, sty, sc.affine, sc.tolerance, mode, poff)
    out = torch.empty((total, width), dtype=torch.float32, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2

    def step(ev=None):
        if ev:
            ev[0].record(stream)
        B.sx_count(ctx, tags, pts, sty, sc.affine, sc.tolerance, mode, poff, want_total=False)
        if ev:
            ev[1].record(stream)
        B.sx_write(ctx, out, total)
        if ev:
            ev[2].record(stream)

    for _ in range(max(args.warmup, 3)):
        flush.fill_(1)
        step()
    torch.cuda.synchronize()
    assert B.sx_last_error(ctx) == 0

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    launches0 = B.sx_launch_count(ctx)
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    for k in range(args.steps):
        flush.fill_(k & 0xff)  # L2 flush between timed steps (outside the event brackets)
        step(evs[k])
    barrier()
    clocks = sampler.stop()
    launches = B.sx_launch_count(ctx) - launches0
    assert B.sx_last_error(ctx) == 0
    t_count = sum(e[0].elapsed_time(e[1]) for e in evs) * 1e-3
    t_write = sum(e[1].elapsed_time(e[2]) for e in evs) * 1e-3
    t_total = sum(e[0].elapsed_time(e[2]) for e in evs) * 1e-3
    t_total = max_over_ranks(t_total, world, dev)

    # ---- end to end through the host-buffer entry point (pinned host memory, copies inside the timed region)
    htags, hpts, hsty = B.scene_to_torch(sc, pin=True)
    hout = torch.empty((total, width), dtype=torch.float32).pin_memory()
    hpoff = torch.empty(n_paths + 1, dtype=torch.int64).pin_memory()
    e2e_steps = max(3, min(args.steps, 10))
    B.stroke_expand_host(ctx, htags, hpts, hsty, sc.affine, sc.tolerance, mode, hout, hpoff)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        m = B.stroke_expand_host(ctx, htags, hpts, hsty, sc.affine, sc.tolerance, mode, hout, hpoff)
    torch.cuda.synchronize()
    t_e2e = time.perf_counter() - t0
    assert m == total
    t_e2e = max_over_ranks(t_e2e, world, dev)
    h2d = tags.numel() + pts.numel() * 4 + sty.numel()
    d2h = total * width * 4 + (n_paths + 1) * 8

    if rank == 0:
        peak, peak_src = load_peaks()
        # algorithmic bytes of the dominant kernel (write): the streams it must read + the records it must write
        alg_bytes = tags.numel() + pts.numel() * 4 + sty.numel() + total * width * 4
        ach = alg_bytes / (t_write / args.steps) / 1e9
        alg_step = alg_bytes + (n_paths + 1) * 8  # + the per-path offsets written by the allocation scan
        line = {"metric": METRIC, "value": job_throughput(n_seg, args.steps, world, t_total), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": 1e3 * t_total / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": args.workload, "segments": n_seg, "paths": n_paths, "records": int(total),
                           "mode": "arc" if mode else "line", "tolerance": float(sc.tolerance), "l2": "flushed between steps (256 MiB fill)",
                           "parallelism": "replicas only" if world > 1 else "single GPU"},
                "output_records_per_s": job_throughput(total, args.steps, world, t_total),
                "kernel_ms": {"scan+count+alloc_scan": 1e3 * t_count / args.steps, "write": 1e3 * t_write / args.steps},
                "gpu_launches": int(launches), "clocks": clocks,
                "e2e": {"value": job_throughput(n_seg, e2e_steps, world, t_e2e), "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                        "ms_per_step": 1e3 * t_e2e / e2e_steps},
                "roofline": {"kernel": "write pass (d): k_write_pieces + k_write_segments, timed together around sx_write",
                             "bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                             "traffic": NCU_TRAFFIC.get(args.workload) if args.paths is None else None,
                             "peak_source": peak_src, "algorithmic_bytes_per_launch": int(alg_bytes),
                             "whole_step": {"achieved": alg_step / (t_total / args.steps) / 1e9, "frac": alg_step / (t_total / args.steps) / 1e9 / peak,
                                            "algorithmic_bytes": int(alg_step)},
                             "fp32_issue_peak_lane_ops_per_s": 148 * 128 * 1.965e9,
                             "note": "measured regime is FP32/ALU issue, not HBM (DESIGN.md section 8, profiles/)"}}
        # ---- the oracle timed beside it on this box's host cores (single thread), bounded sample
        if world == 1 and not args.no_cpu_baseline:
            npaths = REF_SAMPLE_PATHS[args.workload] * 5
            sub = make_scene(args.workload, n_paths=min(npaths, n_paths))
            dt, r = time_oracle(sub, mode, reps=3)
            line["cpu_baseline"] = {"value": sub.n_segments / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
                                    "sample": f"first {sub.n_paths} paths of {args.workload} ({sub.n_segments} segments -> {r.n_rec} records), best of 3"}
        print(json.dumps(line), flush=True)
    B.sx_destroy(ctx)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c4", choices=sorted(MODE_OF))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--mode", default=None, choices=["line", "arc"], help="override the workload's output mode")
    ap.add_argument("--paths", type=int, default=None, help="profiling only: shrink the workload to this many paths")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
