#!/usr/bin/env python
"""bench.py -- throughput of the stroke-expansion hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c4|c5|c3|c2|c1] [--mode line|arc|refined] [--impl ours|reference]

A step is one pass of the whole hot path -- kernels (a) tag scan, (b) count pass, (c) allocation scan, (d) the four
writers -- over one synthetic scene (default: config 4, the CAD-scale scene BASELINE.json's target is quoted on:
1,000,000 segments, arc output, tolerance 0.1), through the C-ABI call `stroke_expand_into`.  `value` is input segments
per second with the streams resident in HBM, device-timed with CUDA events on the launching stream (L2 flushed between
steps); `e2e` is the same metric through the host-buffer C-ABI call with the H2D / D2H copies inside the timed region.
`roofline` is the whole step (algorithmic bytes over the device-timed step against the measured HBM peak; the dominant
kernel is named by the library's own per-kernel events); `roofline.whole_step` is T_roof / T_step with the three ceilings of SURVEY 8(d)
(algorithmic bytes / measured HBM bandwidth, FP32 lane-operations / measured FFMA issue rate, MUFU operations / measured
MUFU rate), the unit counts taken from the instrumented oracle on a sample of the scene.  `--impl reference` times the CPU
oracle instead.  Prints ONE JSON line (rank 0).  With --gpus N > 1 and no torchrun environment, bench.py starts the N
replicas itself (torch.distributed.run, one process per GPU).
"""
from __future__ import annotations

import argparse
import json
import multiprocessing as mp
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "input path segments/sec expanded (device-timed)"
UNIT = "segments/s"
MODE_NAME = {0: "line", 1: "arc", 2: "line-refined"}
MODE_OF = {"c3": 0, "c4": 1, "c5": 0, "c1": 0, "c2": 0}
# whole-step dram__bytes_read.sum + dram__bytes_write.sum per step from the committed `ncu --set full` captures
# (profiles/r2_counters.md names the command and the commit of each); None = not captured for that workload / mode
NCU_TRAFFIC = {"c4-arc": 525.9e6, "c5-line": 23232e6, "c5-arc": 24513e6, "c3-line": 74.3e6}
NCU_TRAFFIC_SOURCE = "profiles/r2_counters.md"
REF_SAMPLE_PATHS = {"c4": 20000, "c5": 1000, "c3": 20000, "c1": 256, "c2": 2000}
# issue slots (FMA = 1) and special-function operations per unit of the method's own work
SLOTS = {"fit_iter": (110, 7), "piece": (60, 2), "range_line": (30, 5), "range_arc": (12, 2), "vertex_line": (65, 4),
         "record_arc": (55, 3), "vertex_evolute": (60, 4), "join": (40, 4), "round_vertex": (6, 0), "cap": (20, 2)}
FP32_THEORETICAL = 148 * 128 * 1.965e9


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML; start() returns once the first sample is in."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop_evt, self._ready, self._mark = threading.Event(), threading.Event(), None

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = int(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
            names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                     "hw_power_brake_slowdown": 0x80, "sync_boost": 0x10, "applications_clocks_setting": 0x2}
            while not self._stop_evt.is_set():
                mhz = int(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(h))
                if self._mark is not None:
                    self.samples.append(mhz)
                    for k, bit in names.items():
                        if r & bit:
                            self.reasons.add(k)
                self._ready.set()
                time.sleep(0.001)
        except Exception as e:  # no NVML: report that, never fake numbers
            self.reasons.add(f"nvml_unavailable:{type(e).__name__}")
            self._ready.set()

    def begin(self):
        """Start the thread (before the warm-up) and wait for NVML to answer."""
        self.start()
        self._ready.wait(timeout=10)

    def mark(self):
        """Samples taken from now on belong to the timed region."""
        self._mark = time.perf_counter()

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


DASH = None   # --dash: (pattern in px, phase) applied to every path
DASH_PATTERN = ([30.0, 12.0, 6.0, 12.0], 7.0)


def make_scene(workload, n_paths=None):
    from paper_2405_00127_b200 import scenes as S
    sc = S.make(workload, n_paths=n_paths)
    return S.with_dash(sc) if DASH else sc


# ---------------------------------------------------------------- the oracle on the host cores
def _oracle_chunk(job):
    import oracle
    tags, points, styles, affine, tol, mode, dash = job
    t0 = time.perf_counter()
    r = oracle.expand(tags, points, styles, affine, tol, mode, dash=dash[0] if dash else None, phase=dash[1] if dash else 0.0)
    return time.perf_counter() - t0, r.n_rec, r.stats


def oracle_jobs(sc, mode, n_chunks):
    """The scene cut into n_chunks runs of whole paths (paths are independent units)."""
    from paper_2405_00127_b200 import scenes as S
    bounds = np.linspace(0, sc.n_paths, n_chunks + 1).astype(int)
    jobs = []
    for a, b in zip(bounds[:-1], bounds[1:]):
        if b > a:
            sub, _ = S.subset_paths(sc, np.arange(a, b))
            jobs.append((sub.tags, sub.points, sub.styles, sub.affine, float(sub.tolerance), mode, DASH))
    return jobs


def time_oracle(jobs, pool=None, reps=1):
    """Wall-clock seconds of the oracle over the jobs (oracle_jobs: the scene cut into runs of whole paths, one per
    process of the pool), best of reps; records; summed unit counts."""
    best, out = None, None
    for _ in range(reps):
        t0 = time.perf_counter()
        res = [_oracle_chunk(j) for j in jobs] if pool is None else pool.map(_oracle_chunk, jobs)
        dt = time.perf_counter() - t0
        if best is None or dt < best:
            best, out = dt, res
    stats = {}
    for _, _, st in out:
        for k, v in st.items():
            stats[k] = stats.get(k, 0) + v
    return best, sum(r[1] for r in out), stats


def make_pool(cores):
    if cores <= 1:
        return None
    pool = mp.get_context("fork").Pool(cores)
    pool.map(abs, range(cores))  # the workers are up before anything is timed
    return pool


def run_reference(args):
    """The oracle, as it stands, on all host cores (one process per core over runs of whole paths); each step a bounded
    sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    oracle.build()
    mode = MODE_OF[args.workload] if args.mode is None else {"line": 0, "arc": 1, "refined": 2}[args.mode]
    cores = os.cpu_count() or 1
    npaths = REF_SAMPLE_PATHS[args.workload] * (4 if cores >= 8 else 1)
    sc = make_scene(args.workload, n_paths=npaths)
    pool = make_pool(cores)
    jobs = oracle_jobs(sc, mode, cores)
    for _ in range(max(args.warmup, 1)):
        time_oracle(jobs, pool)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _, n_rec, _ = time_oracle(jobs, pool)
    dt = time.perf_counter() - t0
    if pool is not None:
        pool.close()
    value = sc.n_segments * args.steps / dt
    sample = f"first {sc.n_paths} paths of {args.workload} ({sc.n_segments} segments -> {n_rec} records) per step, {cores} processes over runs of whole paths"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": args.workload, "mode": MODE_NAME[mode], "tolerance": float(sc.tolerance), "sample": sample, **({"dash": list(DASH[0]), "dash_phase": DASH[1]} if DASH else {})},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def unit_work(stats, kinds, mode, scale):
    """I_fp32, I_mufu of SURVEY 8(d) from the instrumented oracle's unit counts (scaled from the sample to the scene)."""
    k3 = kinds & 7
    n_join_outer, n_cap = int((k3 == 4).sum()), int((k3 == 6).sum())
    joins = stats["joins"] // 2
    units = {"fit_iter": stats["fit_iters"], "piece": stats["pieces"],
             "range_arc" if mode == 1 else "range_line": stats["ranges_reg"] + stats["ranges_sup"],
             "record_arc" if mode == 1 else "vertex_line": stats["rec_offset"],
             "vertex_evolute": stats["rec_evolute"] // 2 + stats["rec_connector"] // 2,
             "join": joins, "cap": stats["caps"],
             "round_vertex": max(0, n_join_outer - joins) + max(0, n_cap - stats["caps"])}
    i_fp32 = sum(SLOTS[k][0] * v for k, v in units.items()) * scale
    i_mufu = sum(SLOTS[k][1] * v for k, v in units.items()) * scale
    return i_fp32, i_mufu, {k: int(v * scale) for k, v in units.items()}


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

    mode = MODE_OF[args.workload] if args.mode is None else {"line": 0, "arc": 1, "refined": 2}[args.mode]
    sc = make_scene(args.workload, n_paths=args.paths)  # replicas only: every rank expands the whole scene
    n_seg, n_paths = sc.n_segments, sc.n_paths
    tags, pts, sty = B.scene_to_torch(sc, device=dev)
    width = 8 if mode == 1 else 4
    sampler = ClockSampler(local)
    sampler.begin()
    issue = B.sx_measure_issue_peaks(local)
    ctx = B.sx_create(local)
    if DASH:
        B.sx_set_dash(ctx, DASH[0], DASH[1])
    stream = torch.cuda.current_stream()
    poff = torch.empty(n_paths + 1, dtype=torch.int64, device=dev)
    total = B.sx_count(ctx, tags, pts, sty, sc.affine, sc.tolerance, mode, poff)
    out = torch.empty((total, width), dtype=torch.float32, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2

    def step():
        # the call a user makes when the capacity is known: asynchronous, no host round trip
        B.stroke_expand_into(ctx, tags, pts, sty, sc.affine, sc.tolerance, mode, out, poff, want_total=False)

    warm = max(args.warmup, 3)
    for _ in range(warm):
        flush.fill_(1)
        step()
    torch.cuda.synchronize()
    assert B.sx_last_error(ctx) == 0
    assert int(poff[-1].item()) == total

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(args.steps)]
    launches0 = B.sx_launch_count(ctx)
    barrier()
    sampler.mark()
    for k in range(args.steps):
        flush.fill_(k & 0xff)  # L2 flush between timed steps (outside the event brackets)
        evs[k][0].record(stream)
        step()
        evs[k][1].record(stream)
    barrier()
    launches = B.sx_launch_count(ctx) - launches0
    assert B.sx_last_error(ctx) == 0
    t_total = sum(e[0].elapsed_time(e[1]) for e in evs) * 1e-3
    t_total = max_over_ranks(t_total, world, dev)
    # keep the GPU under the same load until the sampler has seen it (short workloads finish between two NVML polls)
    t_end = time.perf_counter() + 0.25
    while len(sampler.samples) < 3 and time.perf_counter() < t_end:
        step()
        torch.cuda.synchronize()
    clocks = sampler.stop()
    stats = B.sx_call_stats(ctx)

    # ---- per-kernel durations: the library's own events on the launching stream, one query (sync) per step
    B.sx_set_option(ctx, B.SX_OPT_TIME_KERNELS, 1)
    k_steps = max(3, min(args.steps, 10))
    t_k = np.zeros(4)
    for k in range(k_steps):
        flush.fill_(k & 0xff)
        step()
        t_k += np.array(B.sx_kernel_times(ctx)) * 1e-3
    B.sx_set_option(ctx, B.SX_OPT_TIME_KERNELS, 0)
    t_k /= k_steps
    t_scan, t_count, t_alloc, t_write = (float(x) for x in t_k)

    # ---- the one-shot call with an unknown record count: count pass, host read of the total, allocation, write pass
    o_steps = max(3, min(args.steps, 5))
    B.stroke_expand(ctx, tags, pts, sty, sc.affine, sc.tolerance, mode)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(o_steps):
        rec1, _ = B.stroke_expand(ctx, tags, pts, sty, sc.affine, sc.tolerance, mode)
    torch.cuda.synchronize()
    t_one = (time.perf_counter() - t0) / o_steps
    assert rec1.shape[0] == total
    del rec1

    # ---- tile binning of the records just written (line mode only), device-timed
    binning = None
    if args.binning and mode != 1:
        ext = float(sc.points.max()) + 128.0
        tiles_xy = int(np.ceil(ext / 16.0))
        toff = torch.empty(tiles_xy * tiles_xy + 1, dtype=torch.int32, device=dev)
        try:
            B.sx_bin_lines(ctx, out, tiles_xy, tiles_xy, toff, None)
            pairs = 0
        except B.StrokeExpandError as e:
            pairs = e.needed
        B.sx_last_error(ctx)
        tlines = torch.empty(max(pairs, 1), dtype=torch.int32, device=dev)
        b_evs = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(5)]
        for k in range(8):
            flush.fill_(k)
            if k >= 3:
                b_evs[k - 3][0].record(stream)
            B.sx_bin_lines(ctx, out, tiles_xy, tiles_xy, toff, tlines, want_total=False)
            if k >= 3:
                b_evs[k - 3][1].record(stream)
        torch.cuda.synchronize()
        assert B.sx_last_error(ctx) == 0 and int(toff[-1].item()) == pairs
        t_bin = float(np.mean([e[0].elapsed_time(e[1]) for e in b_evs])) * 1e-3
        b_bytes = 2 * 16 * total + 4 * pairs + 12 * (tiles_xy * tiles_xy + 1)
        binning = {"call": "sx_bin_lines (count, scan, scatter) on the records of this step", "tiles": [tiles_xy, tiles_xy], "pairs": int(pairs),
                   "ms_per_call": 1e3 * t_bin, "records_per_s": total / t_bin, "algorithmic_bytes": int(b_bytes),
                   "achieved_gbs": b_bytes / t_bin / 1e9}

    # ---- end to end through the host-buffer entry point (pinned host memory, copies inside the timed region)
    htags, hpts, hsty = B.scene_to_torch(sc, pin=True)
    hout = torch.empty((total, width), dtype=torch.float32).pin_memory()
    hpoff = torch.empty(n_paths + 1, dtype=torch.int64).pin_memory()
    e2e_steps = max(3, min(args.steps, 10))
    B.stroke_expand_host(ctx, htags, hpts, hsty, sc.affine, sc.tolerance, mode, hout, hpoff)
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
        t_step = t_total / args.steps
        # algorithmic bytes: the streams read once, the records and the path offsets written once
        alg_bytes = tags.numel() + pts.numel() * 4 + sty.numel() + total * width * 4 + (n_paths + 1) * 8
        dominant, t_dom = max((("k_count (count pass: fit, counts, leaf records)", t_count), ("writers (k_write_segments, k_write_simple, k_write_general, k_write_walk)", t_write)), key=lambda kv: kv[1])
        # the path is several kernels and its algorithmic bytes belong to the step as a whole (the count pass reads the streams,
        # the writers write the records): the roofline line is the WHOLE STEP -- algorithmic bytes over the device-timed step --
        # with the dominant kernel named by measured time and the per-kernel durations beside it
        ach = alg_bytes / t_step / 1e9
        key = f"{args.workload}-{MODE_NAME[mode]}"
        line = {"metric": METRIC, "value": job_throughput(n_seg, args.steps, world, t_total), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": warm, "ms_per_step": 1e3 * t_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": args.workload, **({"dash": list(DASH[0]), "dash_phase": DASH[1]} if DASH else {}), "segments": n_seg, "paths": n_paths, "records": int(total),
                           "mode": MODE_NAME[mode], "tolerance": float(sc.tolerance), "l2": "flushed between steps (256 MiB fill)",
                           "call": "stroke_expand_into (tag scan, count pass, allocation scan, writers; asynchronous, no host round trip)",
                           "parallelism": "replicas only" if world > 1 else "single GPU"},
                "output_records_per_s": job_throughput(total, args.steps, world, t_total),
                "kernel_ms": {"k_tag_scan": 1e3 * t_scan, "k_count": 1e3 * t_count, "k_alloc_scan": 1e3 * t_alloc, "writers": 1e3 * t_write,
                              "timed_by": "library events on the launching stream, mean of %d steps" % k_steps},
                "tiles": stats,
                **({"binning": dict(binning, frac_of_hbm_peak=binning["achieved_gbs"] / peak)} if binning else {}),
                "gpu_launches": int(launches), "clocks": clocks,
                "one_shot": {"call": "stroke_expand (count pass, host read of the total, allocation callback, write pass)",
                             "ms_per_call_wall": 1e3 * t_one, "value": n_seg / t_one, "unit": UNIT},
                "e2e": {"value": job_throughput(n_seg, e2e_steps, world, t_e2e), "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                        "ms_per_step": 1e3 * t_e2e / e2e_steps},
                "roofline": {"kernel": "whole step (k_tag_scan, k_count, k_alloc_scan, writers); dominant: %s, %.1f %% of the kernel time" % (dominant, 100 * t_dom / float(t_k.sum())),
                             "bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                             "dominant_kernel_ms": 1e3 * t_dom,
                             "traffic": NCU_TRAFFIC.get(key) if args.paths is None else None, "traffic_source": NCU_TRAFFIC_SOURCE,
                             "peak_source": peak_src, "algorithmic_bytes_per_launch": int(alg_bytes),
                             "bytes_per_segment": alg_bytes / n_seg}}
        # ---- the oracle timed beside it on this box's host cores: one core and all cores, bounded sample; its unit
        # counts give the FP32 / MUFU ceilings of the whole step
        if world == 1 and not args.no_cpu_baseline:
            cores = os.cpu_count() or 1
            npaths = min(REF_SAMPLE_PATHS[args.workload] * 5, n_paths)
            sub = make_scene(args.workload, n_paths=npaths)
            dt1, n_rec, st = time_oracle(oracle_jobs(sub, mode, 1), None, reps=2)
            pool = make_pool(cores)
            dtn, _, _ = time_oracle(oracle_jobs(sub, mode, cores), pool, reps=3)
            if pool is not None:
                pool.close()
            sample = f"first {sub.n_paths} paths of {args.workload} ({sub.n_segments} segments -> {n_rec} records), best of 2 (one core) / 3 (all cores)"
            line["cpu_baseline"] = {"value": sub.n_segments / dtn, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                                    "one_core": {"value": sub.n_segments / dt1, "cores": 1}}
            import oracle
            r = oracle.expand(sub.tags, sub.points, sub.styles, sub.affine, sub.tolerance, mode, dash=DASH[0] if DASH else None, phase=DASH[1] if DASH else 0.0)
            i_fp32, i_mufu, units = unit_work(r.stats, r.kind, mode, n_seg / sub.n_segments)
            ceil = {"hbm_ms": 1e3 * alg_bytes / (peak * 1e9), "fp32_ms": 1e3 * i_fp32 / issue["fp32_ffma"], "mufu_ms": 1e3 * i_mufu / issue["mufu"]}
            bound = max(ceil, key=ceil.get)
            line["roofline"]["whole_step"] = {
                "t_roof_ms": ceil[bound], "t_step_ms": 1e3 * t_step, "frac": ceil[bound] / (1e3 * t_step), "bound": bound.split("_")[0],
                "ceilings_ms": ceil, "i_fp32_lane_ops": i_fp32, "i_mufu_ops": i_mufu, "units": units,
                "r_fp32_measured": issue["fp32_ffma"], "r_fp32_mix_measured": issue["fp32_mix"], "r_fp32_theoretical": FP32_THEORETICAL,
                "r_mufu_measured": issue["mufu"], "slot_table": "SURVEY 8(d)", "units_from": sample}
        print(json.dumps(line), flush=True)
    B.sx_destroy(ctx)
    if world > 1:
        dist.destroy_process_group()


def main():
    global DASH
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c4", choices=sorted(MODE_OF))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--mode", default=None, choices=["line", "arc", "refined"], help="override the workload's output mode (refined: SX_MODE_LINE_REFINED)")
    ap.add_argument("--dash", action="store_true", help="dash every path with the pattern 30-12-6-12 px, phase 7 (SURVEY 8(f)-3: GPU dashing)")
    ap.add_argument("--binning", action="store_true", help="line mode: also time the tile binning of the records (SURVEY 8(f)-4)")
    ap.add_argument("--paths", type=int, default=None, help="profiling only: shrink the workload to this many paths")
    args = ap.parse_args()
    if args.dash:
        DASH = DASH_PATTERN
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # started by hand: become the launcher of N replicas, one process per GPU
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
               "--master-port", str(29500 + os.getpid() % 1000), os.path.abspath(__file__)] + sys.argv[1:]
        sys.exit(subprocess.call(cmd))
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
