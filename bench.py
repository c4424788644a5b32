#!/usr/bin/env python
"""bench.py -- headline benchmark: formal-solution ray-voxel segments*lambda per second on B200.

A "step" is one pass of the whole hot path over one synthetic atmosphere:
dex_build_sparse_grid + dex_build_vlm_mips + dex_mean_intensity (fused HDDA march to J).  The default
workload is BASELINE.json configs[1] (C2: 512x512, 16x16 bricks, 60 % empty, 32 wavelengths, 64
directions, a probe at every voxel, VLM levels 0-3 at relative variance 1e-2).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload C1..C5]

N > 1 (torchrun): every rank solves its own seeded atmosphere of the same size (weak scaling, no
data-path collective -- rays are independent); NCCL is used only for the barrier and
the max-over-ranks of the device time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "formal_solution_ray_voxel_segments_lambda_per_sec"
UNIT = "seg*lambda/s"
ALGO_BYTES = {0: 8.0, 1: 16.0, 2: 8.0, 3: 8.0}   # per seg*lambda: ISO 8 (eta, chi fp32), VELINTERP 16, CAV bg 8
VARIANT_NAME = {0: "iso", 1: "velinterp", 2: "cav", 3: "classic"}
# Core-and-Voigt is bound by plain fp32 arithmetic, not by memory: algorithmic flops (an FMA
# counts 2) per (segment, wavelength, active line) of the fp32 profile evaluation + line sum, and per (segment,
# wavelength) of the segment integral; peak = 148 SMs x 128 fp32 lanes x 2 flop x SM clock.
CAV_FLOPS_PER_LINE_EVAL = 75.0
CAV_FLOPS_PER_SEG_LAMBDA = 25.0
FP32_LANES = 148 * 128


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C2", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--n", type=int, default=None, help="override grid side (reduced-size runs)")
    ap.add_argument("--n-dirs", type=int, default=None)
    ap.add_argument("--n-probes", type=int, default=None, help="seeded probe subset (default: every probe)")
    ap.add_argument("--probe-band", type=float, default=None,
                    help="keep only the probes of a centred band of this fraction of the slowest axis (contiguous, "
                         "coherent subset for profiling)")
    ap.add_argument("--probe-tile", default=None, help="reorder 2D every-voxel probes into WxH tiles, e.g. 8x4")
    ap.add_argument("--lanes", type=int, default=None, help="lanes per ray (1/2/4/8)")
    ap.add_argument("--tile", type=int, default=None, help="tile_probes tuning knob (0/1)")
    ap.add_argument("--cpu-probes", type=int, default=None, help="probes in the oracle (cpu_baseline) sample")
    ap.add_argument("--pipeline", type=int, default=0,
                    help="time the per-iteration rebuild pipeline (dex_mean_intensity_pipelined) with this many "
                         "wavelength batches per stage instead of the whole-spectrum build + march")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def config_dict(wl, args, extra=None):
    c = {
        "workload": f"{wl.name}: {wl.ndim}D {'x'.join(str(d) for d in wl.dims[:wl.ndim])} grid, brick {wl.brick}, "
                    f"{100.0 * (1.0 - float(wl.active.mean())):.0f}% voxels inactive, {wl.n_lambda} wavelengths "
                    f"(batches of {wl.lambda_batch}), {wl.dirs.shape[0]} directions, {wl.probe_pos.shape[0]} probes, "
                    f"variant {VARIANT_NAME[wl.variant]}, VLM max_level {wl.max_level} metric "
                    f"{'relvar' if wl.metric == 1 else 'iod_log'} thr {wl.thr_eta:g}",
        "baseline_config": {"C1": "configs[0]", "C2": "configs[1]", "C3": "configs[2]", "C4": "configs[3]",
                            "C5": "configs[4]"}[wl.name],
        "n_rays": int(wl.probe_pos.shape[0] * wl.dirs.shape[0]),
        "seed": wl.notes.get("seed"),
        "l2": "flushed between timed steps (256 MiB device memset outside the timed events)",
        "parallelism": f"replicas x{args.gpus} (independent atmospheres, no data-path collective)",
    }
    if extra:
        c.update(extra)
    return c


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 8:
                continue
            try:
                sm.append(float(f[1]))
                mx.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def cpu_baseline(wl, n_probes, steps=1):
    """The oracle as it stands, timed on this box's host cores on a bounded sample of the workload."""
    from oracle import oracle as orc
    from workloads.gen import sample_probes
    M = orc.build_mips(wl)
    target_s = 12.0                       # "about 10-30 s of CPU work": a pilot sample sizes the timed one
    total = wl.probe_pos.shape[0]
    n_probes = min(n_probes, total)
    best, segs, pp = None, 0, None
    for attempt in range(3):
        pp = sample_probes(wl.probe_pos, n_probes, 4242)
        best = None
        for _ in range(steps):
            t0 = time.perf_counter()
            res = orc.hdda_march(wl, M, probe_pos=pp)
            dt = time.perf_counter() - t0
            segs = res.segments
            best = dt if best is None else min(best, dt)
        if best >= 0.6 * target_s or n_probes >= total:
            break
        n_probes = min(total, max(n_probes + 1, int(n_probes * target_s / max(best, 1e-3))))
    cores = orc.max_threads()
    return {
        "value": segs * wl.lambda_batch / best, "unit": UNIT, "cores": cores, "kind": "oracle",
        "sample": f"{pp.shape[0]} seeded probes x {wl.dirs.shape[0]} directions x {wl.n_lambda} wavelengths of the same "
                  f"workload ({segs} segments, HDDA+VLM oracle march, OpenMP over probes, {best:.2f} s; mip/level "
                  f"build not timed)",
        "seconds": best,
    }


def run_reference(args):
    """--impl reference: for this tier the reference arm is the oracle on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from workloads import make
    wl = make(args.workload, n=args.n, n_dirs=args.n_dirs, n_probes=args.n_probes)
    n_probes = args.cpu_probes or {"C1": 4096, "C2": 2048, "C3": 256, "C4": 24, "C5": 256}[wl.name]
    from oracle import oracle as orc
    from workloads.gen import sample_probes
    pp = sample_probes(wl.probe_pos, n_probes, 4242)
    M = orc.build_mips(wl)
    times, segs = [], 0
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        res = orc.hdda_march(wl, M, probe_pos=pp)
        dt = time.perf_counter() - t0
        segs = res.segments
        if i >= args.warmup:
            times.append(dt)
    ms = 1e3 * float(np.mean(times))
    value = segs * wl.lambda_batch / (ms * 1e-3)
    cores = orc.max_threads()
    sample = (f"each step = {pp.shape[0]} seeded probes x {wl.dirs.shape[0]} directions x {wl.n_lambda} wavelengths "
              f"({segs} segments) of the workload, oracle HDDA+VLM march on {cores} host threads")
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": config_dict(wl, args, {"l2": "n/a (CPU)"}),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out))


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
        return
    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    import paper_2511_08498_b200 as P
    from workloads import make
    from workloads.gen import SEEDS

    # weak scaling: every rank owns an atmosphere of the same size (its own seed)
    wl = make(args.workload, n=args.n, n_dirs=args.n_dirs, n_probes=args.n_probes,
              seed=P.shard.rank_seed(SEEDS[args.workload], rank))
    if args.probe_band:
        ax = wl.ndim - 1
        n_ax = wl.dims[ax]
        lo, hi = n_ax * (0.5 - args.probe_band / 2), n_ax * (0.5 + args.probe_band / 2)
        keep = (wl.probe_pos[:, ax] >= lo) & (wl.probe_pos[:, ax] < hi)
        wl.probe_pos = np.ascontiguousarray(wl.probe_pos[keep])
    if args.probe_tile and wl.ndim == 2:
        tw, th = (int(v) for v in args.probe_tile.split("x"))
        px = np.floor(wl.probe_pos[:, 0]).astype(np.int64)
        py = np.floor(wl.probe_pos[:, 1]).astype(np.int64)
        key = ((py // th) * (wl.dims[0] // tw) + (px // tw)) * (tw * th) + (py % th) * tw + (px % tw)
        wl.probe_pos = np.ascontiguousarray(wl.probe_pos[np.argsort(key, kind="stable")])
    if args.lanes:
        P.dex_set_lanes_per_ray(args.lanes)
    if args.tile is not None:
        P.dex_set_tuning("tile_probes", args.tile)
    W = wl.lambda_batch
    dw = P.pipeline.upload(wl, dev, non_blocking=False)
    n_probes = wl.probe_pos.shape[0]
    J = torch.empty((n_probes, wl.n_lambda), dtype=torch.float32, device=dev)
    seg = torch.zeros(1, dtype=torch.int64, device=dev)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()

    class _NoMips:
        def destroy(self):
            pass

    def step():
        grid = P.pipeline.build_grid(dw)
        if args.pipeline > 0:              # stage s+1's mips are built while stage s is marched
            P.pipeline.mean_intensity_pipelined(dw, grid, args.pipeline, J=J, segment_count=seg)
            return grid, _NoMips()
        mips = P.pipeline.build_mips(dw, grid)
        P.pipeline.mean_intensity(dw, grid, mips, J=J, segment_count=seg)
        return grid, mips

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 0)):
        g, m = step()
        torch.cuda.synchronize()
        m.destroy(); g.destroy()

    clocks = ClockSampler(local)
    P.dex_pool_high_water(reset=True)
    P.dex_march_timing_read(reset=True)
    P.dex_march_timing_enable(True)
    seg.zero_()
    launches0 = P.dex_launch_count()
    barrier()
    clocks.start()
    t_wall0 = time.perf_counter()
    evs = []
    for _ in range(args.steps):
        flush.zero_()                      # L2 flush, outside the timed events
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        g, m = step()
        m.destroy(); g.destroy()           # stream-ordered release into the library's pool: the next step reuses it
        b.record(stream)
        evs.append((a, b))
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clk = clocks.stop()
    launches = P.dex_launch_count() - launches0
    pool_high = P.dex_pool_high_water()
    P.dex_march_timing_enable(False)
    march_ms, march_n = P.dex_march_timing_read(reset=True)
    line_segs = P.dex_march_work_read(reset=True)
    step_ms = [a.elapsed_time(b) for a, b in evs]
    total_ms = float(sum(step_ms))
    segs_total = int(seg.item())
    max_ms, all_segs = P.shard.job_totals(total_ms, segs_total, dev)      # max over ranks, sum over ranks
    value = all_segs * W / (max_ms * 1e-3)

    # end to end through the public API with HOST (pinned) buffers: H2D + build + march + D2H of J per step
    e2e = None
    if not args.no_e2e:
        pinned = P.pipeline.pin(wl)
        # the caller's result buffer: pinned once, reused every step (allocating and pinning 33.5 MB per call costs
        # 4.5 ms on C2; the D2H copy of J into it stays inside the timed region)
        J_host = torch.empty((n_probes, wl.n_lambda), dtype=torch.float32).pin_memory()
        P.pipeline.solve_J_from_host(wl, dev, pinned, J_host)    # warm-up
        torch.cuda.synchronize()
        e_t, e_seg, h2d, d2h = 0.0, 0, 0, 0
        n_e2e = max(1, min(args.steps, 3))
        for _ in range(n_e2e):
            barrier()
            t0 = time.perf_counter()
            _, nseg, h2d, d2h = P.pipeline.solve_J_from_host(wl, dev, pinned, J_host)
            torch.cuda.synchronize()
            e_t += time.perf_counter() - t0
            e_seg += nseg
        e_t_max, e_seg_all = P.shard.job_totals(e_t, e_seg, dev)
        e2e = {"value": e_seg_all * W / e_t_max, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "steps": n_e2e,
               "timing": "host wall clock around ONE dex_mean_intensity_host call (C ABI, pinned host buffers in, pinned host J "
                         "out: H2D + grid build + mips build + fused march + D2H inside), max over ranks"}

    if rank == 0:
        peak, peak_src = peaks()
        seg_per_launch = segs_total / max(1, march_n)
        algo_bytes = ALGO_BYTES[wl.variant] * seg_per_launch * W
        march_avg_ms = march_ms / max(1, march_n)
        achieved = algo_bytes / (march_avg_ms * 1e-3) / 1e9 if march_avg_ms > 0 else 0.0
        traffic = None
        tp = os.path.join(ROOT, "profiles", "traffic.csv")      # ncu dram__bytes_{read,write}.sum per launch
        if os.path.exists(tp):
            import csv
            with open(tp) as f:
                for row in csv.DictReader(f):
                    if row["workload"] == wl.name:
                        traffic = int(row["dram_bytes_read"]) + int(row["dram_bytes_write"])
        roof = {
            "bound": "hbm", "kernel": "dex_march_kernel (fused HDDA march + angular reduction)",
            "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
            "peak_source": peak_src,
            "note": f"achieved = ALGORITHMIC bytes ({ALGO_BYTES[wl.variant]:g} B per segment*lambda for "
                    f"{VARIANT_NAME[wl.variant]}) / march-kernel time from CUDA "
                    "events on the launching stream; cells are revisited by ~1e2-1e3 rays, so the working set is "
                    "L1/L2-resident and this effective figure is not DRAM traffic (see DESIGN.md)",
            "kernel_ms_per_launch": march_avg_ms, "kernel_share_of_step": march_ms / total_ms if total_ms else None,
        }
        if wl.variant in (2, 3) and march_avg_ms > 0:
            # ALU-bound variant: report against the fp32 FMA peak at the clock sampled during the run
            flops = (CAV_FLOPS_PER_LINE_EVAL * line_segs * W + CAV_FLOPS_PER_SEG_LAMBDA * segs_total * W) / max(1, march_n)
            mhz = clk.get("sm_mhz") or clk.get("sm_max_mhz") or 1965.0
            alu_peak = FP32_LANES * 2 * mhz * 1e6 / 1e12
            ach = flops / (march_avg_ms * 1e-3) / 1e12
            roof.update({
                "bound": "alu", "achieved": ach, "peak": alu_peak, "unit": "TFLOP/s", "frac": ach / alu_peak,
                "peak_source": f"derived: 148 SMs x 128 fp32 lanes x 2 flop x {mhz:.0f} MHz (SM clock sampled during "
                               "the timed region); DESIGN.md section 6",
                "hbm_effective_gbs": achieved,
                "line_profile_evaluations_per_launch": line_segs * W / max(1, march_n),
                "note": f"achieved = ALGORITHMIC fp32 flops ({CAV_FLOPS_PER_LINE_EVAL:g} per segment*lambda*active line "
                        f"for the profile + line sum, {CAV_FLOPS_PER_SEG_LAMBDA:g} per segment*lambda for the integral; "
                        "the library counts segments x active lines) / march-kernel time from CUDA events",
            })
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": max_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": config_dict(wl, args, {"lanes_per_ray": args.lanes or ("auto: 8" if wl.probe_pos.shape[0] < 148 * 128 else "auto: 1"),
                                             "segments_per_step": segs_total // max(1, args.steps),
                                             "path": (f"rebuild pipeline, {args.pipeline} batch(es) per stage"
                                                      if args.pipeline > 0 else "whole-spectrum build + march"),
                                             "library_device_bytes_high_water": int(pool_high)}),
            "clocks": clk,
            "e2e": e2e,
            "gpu_launches": int(launches),
            "roofline": roof,
            "wall_s_timed_region": t_wall,
        }
        if not args.no_cpu_baseline:
            ncpu = args.cpu_probes or {"C1": 4096, "C2": 2048, "C3": 256, "C4": 24, "C5": 256}[wl.name]
            out["cpu_baseline"] = cpu_baseline(wl, ncpu)
            out["cpu_baseline"].pop("seconds", None)
        print(json.dumps(out))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
