#!/usr/bin/env python
"""bench.py -- headline benchmark: formal-solution ray-voxel segments*lambda per second on B200.

A "step" is one pass of the whole hot path over one synthetic atmosphere:
dex_build_sparse_grid + dex_build_vlm_mips + dex_mean_intensity (fused HDDA march to J).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload C1..C5]
                  [--configs C1,C2,...|none] [--shard replicas|probes]

BASELINE.json's `metric` names no config, so the headline (`value`, `ms_per_step`, `roofline`, `e2e`,
`cpu_baseline` at the top level of the JSON line) is quoted on the largest single-GPU configuration: C4
(configs[3], 1024x1024, Core-and-Voigt, 208 wavelengths x 128 directions, 8.7e11 segments and ~7 s per
step), timed for EXACTLY --steps steps after --warmup warm-up steps (20 + 5 take three minutes).  The same
process then measures every other BASELINE config (own clock sample, own roofline / e2e / cpu_baseline)
and prints each as its own JSON line {"per_config": "C1", ...} BEFORE the final headline line; the
headline line's `config.all_configs` repeats every config's step time, value, e2e and roofline fraction in
a few numbers, so that one line alone carries C1-C5.  The default run (5 + 3 steps) takes three minutes.

N > 1 (torchrun): `--shard replicas` (default): every rank solves its own seeded atmosphere of the same
size (weak scaling, no data-path collective -- rays are independent); NCCL is used only for
the barrier and the max-over-ranks of the device time.  `--shard probes`: ONE atmosphere replicated on
every rank, the probes split in contiguous ranges (shard.probe_range), J all-gathered over NCCL
(shard.gather_J) inside the timed region (strong scaling).
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
CONFIGS = ("C1", "C2", "C3", "C4", "C5")
HEADLINE = "C4"
BASELINE_CONFIG = {"C1": "configs[0]", "C2": "configs[1]", "C3": "configs[2]", "C4": "configs[3]", "C5": "configs[4]"}
VARIANT_NAME = {0: "iso", 1: "velinterp", 2: "cav", 3: "classic"}
# ALGORITHMIC work per unit (restated in DESIGN.md section 6)
ALGO_BYTES = {0: 8.0, 1: 16.0, 2: 8.0, 3: 8.0}   # bytes per seg*lambda: ISO 8 (eta, chi fp32), VELINTERP 16, CAV bg 8
# fp32 flops (an FMA counts 2) per seg*lambda of the segment integral (1 mul, 1 ex2, ~6 FMA), of the two velocity-bin
# lerps of VELINTERP, and per segment of the HDDA stepping (~25 int / fp32 operations, shared by the W wavelengths)
FLOPS_INTEGRAL = 14.0
FLOPS_VEL_LERP = 6.0
FLOPS_HDDA_PER_SEGMENT = 25.0
# Core-and-Voigt: fp32 profile evaluation + line sum per (segment, wavelength, active line), integral per (segment, wavelength)
CAV_FLOPS_PER_LINE_EVAL = 75.0
CAV_FLOPS_PER_SEG_LAMBDA = 25.0
MUFU_PER_SM_PER_CLK = 16.0      # ex2 results per SM per clock (4 SMSPs x 4 lanes; Blackwell guide)
N_SM = 148
# per-config caps on (warm-up, timed, e2e) steps when the config is NOT the headline: C4 is seconds per step
STEP_CAPS = {"C4": (0, 1, 1)}
# end-to-end steps and steps of the single-direction alternative per config (default: min(steps, 3)); C4: 7 s each
E2E_STEPS = {"C4": 2}
ALT_STEPS = {"C4": 1}
CPU_PROBES = {"C1": 4096, "C2": 2048, "C3": 128, "C4": 24, "C5": 256}
_HOST_THREADS = None


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=HEADLINE, choices=list(CONFIGS), help="headline config")
    ap.add_argument("--configs", default=None,
                    help="comma list of the configs measured into per_config (default: all five at N=1 in the default "
                         "shape, only the headline otherwise; 'none' = headline only)")
    ap.add_argument("--shard", default="replicas", choices=["replicas", "probes"])
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
    ap.add_argument("--memo-budget-mb", type=int, default=None,
                    help='"memo_budget_mb" tuning knob: cap on the memoised march\'s per-direction records (MB)')
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def traffic_row(name):
    """ncu dram__bytes_{read,write}.sum per march launch from the builder-run captures summarised in profiles/."""
    tp = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(tp):
        return None
    import csv
    with open(tp) as f:
        for row in csv.DictReader(f):
            if row["workload"] == name:
                return row
    return None


def config_dict(wl, args, extra=None):
    c = {
        "workload": f"{wl.name}: {wl.ndim}D {'x'.join(str(d) for d in wl.dims[:wl.ndim])} grid, brick {wl.brick}, "
                    f"{100.0 * (1.0 - float(wl.active.mean())):.0f}% voxels inactive, {wl.n_lambda} wavelengths "
                    f"(batches of {wl.lambda_batch}), {wl.dirs.shape[0]} directions, {wl.probe_pos.shape[0]} probes, "
                    f"variant {VARIANT_NAME[wl.variant]}, VLM max_level {wl.max_level} metric "
                    f"{'relvar' if wl.metric == 1 else 'iod_log'} thr {wl.thr_eta:g}",
        "baseline_config": BASELINE_CONFIG[wl.name],
        "n_rays": int(wl.probe_pos.shape[0] * wl.dirs.shape[0]),
        "seed": wl.notes.get("seed"),
        "l2": "flushed between timed steps (256 MiB device memset outside the timed events)",
        "parallelism": (f"replicas x{args.gpus} (independent atmospheres, no data-path collective)" if args.shard == "replicas"
                        else f"probes split over {args.gpus} ranks, one atmosphere replicated, all-gather of J (NCCL)"),
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


def oracle_sample(wl):
    """The workload restricted to ONE wavelength batch (pure column selection, workloads.gen.batch_workload): the
    oracle's numpy mip build over every batch of a BASELINE-size grid takes minutes.  The oracle evaluates the line
    profiles per segment, so its seg*lambda/s falls with the number of active lines of the batch (the GPU's memoised
    march does not); the batch taken is the one nearest the middle of the spectrum among those with the MEDIAN number
    of active lines, and the sample string says how the batches are distributed."""
    from workloads.gen import batch_workload
    if wl.n_batch <= 1:
        return wl, "all wavelengths"
    mid = wl.n_batch // 2
    if wl.active_lines is None:
        b, lines = mid, ""
    else:
        n_act = (np.asarray(wl.active_lines) >= 0).sum(axis=1)
        med = int(np.sort(n_act)[len(n_act) // 2])
        cand = np.flatnonzero(n_act == med)
        b = int(cand[np.argmin(np.abs(cand - mid))])
        hist = np.bincount(n_act)
        lines = (f", {med} active line(s) -- the median; batches with 0/1/2/.. active lines: "
                 f"{'/'.join(str(int(v)) for v in hist)}; the oracle's rate falls with the line count")
    sub, _ = batch_workload(wl, [b])
    return sub, f"wavelength batch {b} of {wl.n_batch} ({wl.lambda_batch} wavelengths{lines})"


def cpu_baseline(wl, n_probes, target_s=10.0, one_thread_s=4.0):
    """The oracle as it stands, timed on this box's host cores on a bounded sample of the workload: all threads, and
    one thread on a proportionally smaller sample."""
    from oracle import oracle as orc
    from workloads.gen import sample_probes
    sub, which = oracle_sample(wl)
    M = orc.build_mips(sub)
    global _HOST_THREADS          # read once: a one-thread march leaves OpenMP (and max_threads()) at one thread
    if _HOST_THREADS is None:
        _HOST_THREADS = orc.max_threads()
    cores = _HOST_THREADS
    total = wl.probe_pos.shape[0]
    n_probes = min(n_probes, total)
    best, segs, pp = None, 0, None
    for attempt in range(3):      # a pilot sample sizes the timed one
        pp = sample_probes(wl.probe_pos, n_probes, 4242)
        t0 = time.perf_counter()
        res = orc.hdda_march(sub, M, probe_pos=pp, n_threads=cores)
        best = time.perf_counter() - t0
        segs = res.segments
        if best >= 0.6 * target_s or n_probes >= total:
            break
        n_probes = min(total, max(n_probes + 1, int(n_probes * target_s / max(best, 1e-3))))
    out = {
        "value": segs * wl.lambda_batch / best, "unit": UNIT, "cores": cores, "kind": "oracle",
        "sample": f"{pp.shape[0]} seeded probes x {wl.dirs.shape[0]} directions x {which} of the same workload "
                  f"({segs} segments, HDDA+VLM oracle march, OpenMP over probes, {best:.2f} s; mip/level build not timed)",
    }
    if one_thread_s > 0 and cores > 1:
        n1 = max(1, int(pp.shape[0] * one_thread_s / max(best, 1e-3) / cores))
        p1 = sample_probes(wl.probe_pos, min(n1, total), 4243)
        t0 = time.perf_counter()
        r1 = orc.hdda_march(sub, M, probe_pos=p1, n_threads=1)
        dt = time.perf_counter() - t0
        out["one_thread"] = {"value": r1.segments * wl.lambda_batch / dt, "unit": UNIT, "cores": 1,
                             "sample": f"{p1.shape[0]} probes, {r1.segments} segments, {dt:.2f} s"}
    return out


def run_reference(args):
    """--impl reference: for this tier the reference arm is the oracle on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from workloads import make
    wl = make(args.workload, n=args.n, n_dirs=args.n_dirs, n_probes=args.n_probes)
    n_probes = args.cpu_probes or {"C1": 4096, "C2": 2048, "C3": 512, "C4": 48, "C5": 1024}[wl.name]
    from oracle import oracle as orc
    from workloads.gen import sample_probes
    pp = sample_probes(wl.probe_pos, n_probes, 4242)
    sub, which = oracle_sample(wl)
    M = orc.build_mips(sub)
    times, segs = [], 0
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        res = orc.hdda_march(sub, M, probe_pos=pp)
        dt = time.perf_counter() - t0
        segs = res.segments
        if i >= args.warmup:
            times.append(dt)
    ms = 1e3 * float(np.mean(times))
    value = segs * wl.lambda_batch / (ms * 1e-3)
    cores = orc.max_threads()
    sample = (f"each step = {pp.shape[0]} seeded probes x {wl.dirs.shape[0]} directions x {which} "
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


class Bench:
    """One process (one rank): measures configs one after the other on its GPU."""

    def __init__(self, args):
        import torch
        import torch.distributed as dist
        self.args, self.torch, self.dist = args, torch, dist
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        if not torch.cuda.is_available():
            raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
        torch.cuda.set_device(self.local)
        self.dev = f"cuda:{self.local}"
        if self.world > 1:
            dist.init_process_group("nccl", device_id=torch.device(self.dev))
        import paper_2511_08498_b200 as P
        self.P = P
        if args.lanes:
            P.dex_set_lanes_per_ray(args.lanes)
        if args.tile is not None:
            P.dex_set_tuning("tile_probes", args.tile)
        if args.memo_budget_mb is not None:
            P.dex_set_tuning("memo_budget_mb", args.memo_budget_mb)
        self.flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=self.dev)
        self.hbm_peak, self.hbm_src = peaks()
        self.fp32_peak = None

    def barrier(self):
        self.torch.cuda.synchronize()
        if self.world > 1:
            self.dist.barrier()
        self.torch.cuda.synchronize()

    def measure_fp32_peak(self):
        """FFMA / FFMA2 microbenchmark inside this run (dex_measure_fp32_peak), clocks sampled around it."""
        if self.fp32_peak is None:
            clocks = ClockSampler(self.local)
            clocks.start()
            best = (0.0, 0.0)
            t0 = time.perf_counter()
            while time.perf_counter() - t0 < 0.5:         # ~30 launches: long enough for a few clock samples
                a, b = self.P.dex_measure_fp32_peak()
                best = (max(best[0], a), max(best[1], b))
            clk = clocks.stop()
            self.fp32_peak = {"ffma_tflops": best[0], "ffma2_tflops": best[1], "sm_mhz": clk.get("sm_mhz"),
                              "nominal_tflops": N_SM * 128 * 2 * (clk.get("sm_mhz") or 1965.0) * 1e6 / 1e12}
        return self.fp32_peak

    def workload(self, name):
        from workloads import make
        from workloads.gen import SEEDS
        args, P = self.args, self.P
        head = name == args.workload
        seed = SEEDS[name] if args.shard == "probes" else P.shard.rank_seed(SEEDS[name], self.rank)
        wl = make(name, n=args.n if head else None, n_dirs=args.n_dirs if head else None,
                  n_probes=args.n_probes if head else None, seed=seed)
        if head and args.probe_band:
            ax = wl.ndim - 1
            n_ax = wl.dims[ax]
            lo, hi = n_ax * (0.5 - args.probe_band / 2), n_ax * (0.5 + args.probe_band / 2)
            keep = (wl.probe_pos[:, ax] >= lo) & (wl.probe_pos[:, ax] < hi)
            wl.probe_pos = np.ascontiguousarray(wl.probe_pos[keep])
        if head and args.probe_tile and wl.ndim == 2:
            tw, th = (int(v) for v in args.probe_tile.split("x"))
            px = np.floor(wl.probe_pos[:, 0]).astype(np.int64)
            py = np.floor(wl.probe_pos[:, 1]).astype(np.int64)
            key = ((py // th) * (wl.dims[0] // tw) + (px // tw)) * (tw * th) + (py % th) * tw + (px % tw)
            wl.probe_pos = np.ascontiguousarray(wl.probe_pos[np.argsort(key, kind="stable")])
        return wl

    def roofline(self, wl, segs_per_launch, line_segs_per_launch, march_avg_ms, march_share, clk):
        W = wl.lambda_batch
        sl = segs_per_launch * W                                  # seg*lambda per launch
        t = march_avg_ms * 1e-3
        pk = self.measure_fp32_peak()
        fp32_peak = max(pk["ffma_tflops"], pk["ffma2_tflops"])
        # the library counts provider evaluations (dex_march_work_read): one per emitted segment when eta, chi are evaluated
        # inside the march, one per (cell, direction, batch) when they are memoised per direction
        evals = line_segs_per_launch * W                          # per wavelength (x active lines for Core-and-Voigt)
        memoised = wl.variant != 0 and line_segs_per_launch < 0.5 * segs_per_launch
        # bytes the launched kernels REQUEST per march region: in the ray loop the variant's nominal bytes per seg*lambda;
        # memoised: the ISO march reads an 8-byte (chi, S) record per seg*lambda, the records kernel writes 8 B per
        # record*lambda and, for velocity interpolation, reads the two 8-byte velocity bins it interpolates between
        # (evals counts record*lambda, times the batch's active lines for Core-and-Voigt: an upper bound there)
        if memoised:
            req_bytes = 8.0 * sl + 8.0 * evals + (16.0 * evals if wl.variant == 1 else 0.0)
            req_what = ("8 B per seg*lambda read by the ISO march + 8 B per memoised record*lambda written"
                        + (" + 16 B of velocity bins read per record*lambda" if wl.variant == 1 else "") + " by the records kernel")
        else:
            req_bytes = ALGO_BYTES[wl.variant] * sl
            req_what = f"{ALGO_BYTES[wl.variant]:g} B per seg*lambda"
        eff_gbs = req_bytes / t / 1e9 if t > 0 else 0.0
        integral = FLOPS_INTEGRAL * sl + FLOPS_HDDA_PER_SEGMENT * segs_per_launch
        if wl.variant in (2, 3):
            flops = CAV_FLOPS_PER_LINE_EVAL * evals + integral
            what = (f"{CAV_FLOPS_PER_LINE_EVAL:g} per fp32 Voigt profile evaluation + line sum (the library counts them: "
                    f"{evals:.3g} per launch, {'memoised per (cell, direction)' if memoised else 'one per segment, wavelength and active line'}), "
                    f"{FLOPS_INTEGRAL:g} per seg*lambda for the segment integral, {FLOPS_HDDA_PER_SEGMENT:g} per segment of HDDA stepping")
            binds = ("instruction issue of the ISO march over per-direction records (the Voigt profiles are evaluated once per cell "
                     "and direction)" if memoised else "fp32 arithmetic (one Voigt profile per segment, wavelength and active line)")
        else:
            flops = integral + FLOPS_VEL_LERP * evals
            what = (f"{FLOPS_INTEGRAL:g} per seg*lambda (segment integral) + {FLOPS_HDDA_PER_SEGMENT:g} per segment of HDDA stepping"
                    + (f" + {FLOPS_VEL_LERP:g} per velocity-bin interpolation ({evals:.3g} per launch, "
                       f"{'memoised per (cell, direction)' if memoised else 'one per seg*lambda'})" if wl.variant == 1 else ""))
            binds = ("instruction issue (fp32 / integer pipes + one MUFU ex2 per seg*lambda); the batch's records are "
                     "L1/L2-resident because every cell is revisited by 1e2-1e3 rays, so DRAM is idle by construction")
        ach = flops / t / 1e12 if t > 0 else 0.0
        mhz = clk.get("sm_mhz") or pk.get("sm_mhz") or 1965.0
        mufu_floor_ms = sl / (N_SM * MUFU_PER_SM_PER_CLK * mhz * 1e6) * 1e3
        roof = {
            "bound": "alu", "kernel": "dex_march_kernel (fused HDDA march + angular reduction)",
            "achieved": ach, "peak": fp32_peak, "unit": "TFLOP/s", "frac": ach / fp32_peak if fp32_peak else None,
            "binds": binds,
            "peak_source": f"measured in this run by dex_measure_fp32_peak: register-resident FFMA {pk['ffma_tflops']:.1f} / packed "
                           f"FFMA2 {pk['ffma2_tflops']:.1f} TFLOP/s at {pk['sm_mhz']} MHz (nominal 148 SMs x 128 lanes x 2 = "
                           f"{pk['nominal_tflops']:.1f})",
            "note": f"achieved = ALGORITHMIC fp32 flops ({what}; FMA = 2) / march-kernel time from CUDA events on the launching stream",
            "kernel_ms_per_launch": march_avg_ms, "kernel_share_of_step": march_share,
            "segments_per_launch": segs_per_launch,
            # the HBM view BASELINE.json's metric asks for: effective (algorithmic bytes / time; exceeds 1 when the reuse
            # is served by L1/L2) and measured DRAM traffic (ncu, builder-run capture named in traffic_source)
            "effective_gbs": eff_gbs, "effective_frac": eff_gbs / self.hbm_peak, "effective_bytes": req_what,
            "hbm_peak_gbs": self.hbm_peak, "hbm_peak_source": self.hbm_src,
            "mufu_floor_ms": mufu_floor_ms, "mufu_floor_frac": mufu_floor_ms / march_avg_ms if march_avg_ms > 0 else None,
            "traffic": None, "dram_gbs": None, "dram_frac": None,
        }
        row = traffic_row(wl.name)
        if row is not None and t > 0:
            tr = int(row["dram_bytes_read"]) + int(row["dram_bytes_write"])
            # the capture may be of a probe subset: scale by the segments of this launch
            cap_segs = float(row.get("segments_in_capture") or 0) or segs_per_launch
            tr_launch = tr * (segs_per_launch / cap_segs)
            roof.update({"traffic": int(tr_launch), "dram_gbs": tr_launch / t / 1e9, "dram_frac": tr_launch / t / 1e9 / self.hbm_peak,
                         "l2_hit_pct": float(row["l2_hit_pct"]) if row.get("l2_hit_pct") else None,
                         "traffic_source": f"profiles/traffic.csv (ncu, builder-run: {row.get('source', '')}); "
                                           "dram_gbs = that traffic / this run's kernel time"})
            if roof["dram_frac"] >= 0.25:
                # the launch moves a quarter of the HBM peak or more (C5: per-direction records read once per segment with
                # little reuse): the binding roofline is HBM.  Algorithmic bytes: the 8 B record per seg*lambda the march reads,
                # plus the 8 B per memoised record*lambda the records kernel writes
                # (evals counts (record, wavelength) pairs, times the active lines of the batch for Core-and-Voigt: one for C5)
                gbs = req_bytes / t / 1e9
                hit = roof.get("l2_hit_pct")
                roof.update({"alu_achieved_tflops": roof["achieved"], "alu_frac": roof["frac"], "alu_peak_tflops": roof["peak"],
                             "bound": "hbm", "achieved": gbs, "peak": self.hbm_peak, "unit": "GB/s", "frac": gbs / self.hbm_peak,
                             "bound_source": "chosen from the builder-run ncu capture in profiles/traffic.csv (DRAM bytes per launch "
                                             "at >= 0.25 of the HBM peak over this run's kernel time), not from a counter read in this run",
                             "binds": "HBM: the ISO march reads one per-direction record per segment with little reuse"
                                      + (f" (L2 hit rate {hit:.1f} % in the capture)" if hit is not None else "")
                                      + (f"; the records of one launch are {8.0 * evals / 1e9:.1f} GB" if memoised else ""),
                             "peak_source": self.hbm_src,
                             "note": f"achieved = ALGORITHMIC bytes ({req_what}) / time of the library's march region "
                                     "(records kernel + march) from CUDA events"})
        return roof

    def measure(self, name, steps, warmup, e2e_steps, want_cpu, cpu_target_s, one_thread_s):
        torch, P, args = self.torch, self.P, self.args
        wl = self.workload(name)
        W = wl.lambda_batch
        all_probes = wl.probe_pos
        lo, hi = 0, all_probes.shape[0]
        if args.shard == "probes" and self.world > 1:
            lo, hi = P.shard.probe_range(all_probes.shape[0], self.world, self.rank)
            wl.probe_pos = np.ascontiguousarray(all_probes[lo:hi])
        dw = P.pipeline.upload(wl, self.dev, non_blocking=False)
        n_probes = wl.probe_pos.shape[0]
        J = torch.empty((n_probes, wl.n_lambda), dtype=torch.float32, device=self.dev)
        seg = torch.zeros(1, dtype=torch.int64, device=self.dev)
        stream = torch.cuda.current_stream()
        gathered = {}

        class _NoMips:
            def destroy(self):
                pass

        def step():
            grid = P.pipeline.build_grid(dw)
            if args.pipeline > 0:              # stage s+1's mips are built while stage s is marched
                P.pipeline.mean_intensity_pipelined(dw, grid, args.pipeline, J=J, segment_count=seg)
                mips = _NoMips()
            else:
                mips = P.pipeline.build_mips(dw, grid)
                P.pipeline.mean_intensity(dw, grid, mips, J=J, segment_count=seg)
            if args.shard == "probes" and self.world > 1:     # the path's one exchange: all-gather of J
                gathered["J"] = P.shard.gather_J(J, all_probes.shape[0])
            return grid, mips

        for _ in range(max(warmup, 0)):
            g, m = step()
            torch.cuda.synchronize()
            m.destroy(); g.destroy()

        clocks = ClockSampler(self.local)
        P.dex_pool_high_water(reset=True)
        P.dex_march_timing_read(reset=True)
        P.dex_march_work_read(reset=True)
        P.dex_march_timing_enable(True)
        seg.zero_()
        launches0 = P.dex_launch_count()
        self.barrier()
        clocks.start()
        t_wall0 = time.perf_counter()
        evs = []
        for _ in range(steps):
            self.flush.zero_()                 # L2 flush, outside the timed events
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            g, m = step()
            m.destroy(); g.destroy()           # stream-ordered release into the library's pool: the next step reuses it
            b.record(stream)
            evs.append((a, b))
        self.barrier()
        t_wall = time.perf_counter() - t_wall0
        clk = clocks.stop()
        launches = P.dex_launch_count() - launches0
        mapping = P.dex_last_march_mapping()     # what the timed marches ran with (same thread)
        pool_high = P.dex_pool_high_water()
        P.dex_march_timing_enable(False)
        march_ms, march_n = P.dex_march_timing_read(reset=True)
        line_segs = P.dex_march_work_read(reset=True)
        step_ms = [a.elapsed_time(b) for a, b in evs]
        total_ms = float(sum(step_ms))
        segs_total = int(seg.item())
        max_ms, all_segs = P.shard.job_totals(total_ms, segs_total, self.dev)      # max over ranks, sum over ranks
        value = all_segs * W / (max_ms * 1e-3)

        shard_check = None
        if args.shard == "probes" and self.world > 1 and self.rank == 0:
            # the gathered J against a single-rank solve of the same atmosphere, bit for bit (rank 0, untimed)
            wl1 = self.workload(name)
            d1 = P.pipeline.upload(wl1, self.dev, non_blocking=False)
            g1 = P.pipeline.build_grid(d1)
            m1 = P.pipeline.build_mips(d1, g1)
            J1 = P.pipeline.mean_intensity(d1, g1, m1)
            torch.cuda.synchronize()
            shard_check = {"gathered_J_equals_single_rank_J_bitwise": bool(torch.equal(J1, gathered["J"]))}
            m1.destroy(); g1.destroy()
            del d1, J1

        # end to end through the public API with HOST (pinned) buffers: H2D + build + march + D2H of J per step
        e2e = None
        if not args.no_e2e and e2e_steps > 0:
            pinned = P.pipeline.pin(wl)
            # the caller's result buffer: pinned once, reused every step (allocating and pinning it per call costs
            # 4.5 ms on C2; the D2H copy of J into it stays inside the timed region)
            J_host = torch.empty((n_probes, wl.n_lambda), dtype=torch.float32).pin_memory()
            if warmup > 1:                     # the timed device steps above have already warmed the library's pool
                P.pipeline.solve_J_from_host(wl, self.dev, pinned, J_host)
                torch.cuda.synchronize()
            e_t, e_seg, h2d, d2h = 0.0, 0, 0, 0
            for _ in range(e2e_steps):
                self.barrier()
                t0 = time.perf_counter()
                _, nseg, h2d, d2h = P.pipeline.solve_J_from_host(wl, self.dev, pinned, J_host)
                torch.cuda.synchronize()
                e_t += time.perf_counter() - t0
                e_seg += nseg
            e_t_max, e_seg_all = P.shard.job_totals(e_t, e_seg, self.dev)
            e2e = {"value": e_seg_all * W / e_t_max, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                   "d2h_bytes_per_step": int(d2h), "steps": e2e_steps, "ms_per_step": 1e3 * e_t_max / e2e_steps,
                   "timing": "host wall clock around ONE dex_mean_intensity_host call (C ABI, pinned host buffers in, pinned host J "
                             "out: H2D + grid build + mips build + fused march + D2H inside), max over ranks"}
            del pinned, J_host

        # Core-and-Voigt in 2D (C4): the alternative the paper itself names for many rays per voxel and direction --
        # single-direction VLM (dex_mean_intensity_single_direction): per direction the Classic fields over
        # the grid, an ISO pyramid of their own, a one-direction ISO march.  Same rays, same J; timed beside the scheme
        # the config prescribes.
        alt = None
        if wl.variant == 2 and wl.ndim == 2 and args.pipeline == 0 and not (args.shard == "probes" and self.world > 1):
            J2 = torch.empty_like(J)
            seg2 = torch.zeros(1, dtype=torch.int64, device=self.dev)
            grid = P.pipeline.build_grid(dw)
            if warmup > 1:
                P.pipeline.mean_intensity_single_direction(dw, grid, J=J2)
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            n_alt = ALT_STEPS.get(name, max(1, min(steps, 3)))
            a.record(stream)
            for _ in range(n_alt):
                P.pipeline.mean_intensity_single_direction(dw, grid, J=J2, segment_count=seg2)
            b.record(stream)
            torch.cuda.synchronize()
            ms_alt = a.elapsed_time(b) / n_alt
            d = ((J2 - J).abs() / J.abs().clamp_min(1e-30)).flatten()
            if d.numel() > (1 << 26):          # kthvalue on a strided 1-in-n sample of the values
                d = d[:: (d.numel() >> 26) + 1].contiguous()
            p999 = float(torch.kthvalue(d, max(1, int(round(0.999 * d.numel())))).values.item()) if d.numel() else 0.0
            alt = {"path": "single-direction VLM (PAPER.md:396): dex_mean_intensity_single_direction, everything inside "
                           "(per-direction Classic fields, ISO mips, one-direction ISO march, J accumulated)",
                   "ms_per_step": ms_alt, "steps": n_alt, "segments_per_step": int(seg2.item()) // n_alt,
                   "value": int(seg2.item()) / n_alt * W / (ms_alt * 1e-3), "unit": UNIT,
                   "p999_rel_diff_of_J_vs_core_and_voigt": p999,
                   "note": "both are approximations of the Classic (level-0, per-voxel velocity) solve; their p99.9 errors "
                           "against it are in profiles/ (accuracy report)"}
            grid.destroy()
            del J2, d

        out = None
        if self.rank == 0:
            march_avg_ms = march_ms / max(1, march_n)
            roof = self.roofline(wl, segs_total / max(1, march_n), line_segs / max(1, march_n), march_avg_ms,
                                 march_ms / total_ms if total_ms else None, clk)
            out = {
                "value": value, "unit": UNIT, "steps": steps, "warmup": warmup, "ms_per_step": max_ms / steps,
                "config": config_dict(wl, args, {"lanes_per_ray": mapping["lanes_per_ray"], "dirs_per_block": mapping["dirs_per_block"],
                                                 "memo_batches_per_group": mapping["memo_batches_per_group"],
                                                 "segments_per_step": segs_total // max(1, steps),
                                                 "path": (f"rebuild pipeline, {args.pipeline} batch(es) per stage"
                                                          if args.pipeline > 0 else "whole-spectrum build + march"),
                                                 "library_device_bytes_high_water": int(pool_high)}),
                "clocks": clk, "e2e": e2e, "gpu_launches": int(launches), "roofline": roof,
                "wall_s_timed_region": t_wall,
            }
            if shard_check:
                out["shard_check"] = shard_check
            if alt:
                out["alt_single_direction"] = alt
            if want_cpu and self.world == 1:
                ncpu = args.cpu_probes or CPU_PROBES[wl.name]
                out["cpu_baseline"] = cpu_baseline(wl, ncpu, cpu_target_s, one_thread_s)
        del dw, J, wl
        torch.cuda.empty_cache()
        return out


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
        return
    B = Bench(args)
    default_shape = (args.n is None and args.n_dirs is None and args.n_probes is None and args.probe_band is None
                     and args.pipeline == 0 and args.shard == "replicas")
    if args.configs is None:
        extra = [c for c in CONFIGS if c != args.workload] if (B.world == 1 and default_shape) else []
    elif args.configs.lower() == "none":
        extra = []
    else:
        extra = [c for c in args.configs.split(",") if c in CONFIGS and c != args.workload]

    head = B.measure(args.workload, args.steps, args.warmup, E2E_STEPS.get(args.workload, max(1, min(args.steps, 3))),
                     not args.no_cpu_baseline, 10.0, 4.0)
    per = {}
    for name in extra:
        cw, cs, ce = STEP_CAPS.get(name, (args.warmup, args.steps, max(1, min(args.steps, 3))))
        r = B.measure(name, min(args.steps, cs), min(args.warmup, cw), ce, not args.no_cpu_baseline, 3.0, 0.0)
        if r is not None:
            if name in STEP_CAPS:
                r["note"] = (f"{r['ms_per_step'] / 1e3:.0f} s per step: {r['warmup']} warm-up + {r['steps']} timed step(s) and "
                             f"{ce} end-to-end step here (a cold first step costs it < 0.1 %: the library's pool is warm from "
                             f"the configs before it); `python bench.py --workload {name}` times it as the headline")
            per[name] = r
    if B.rank == 0:
        out = {
            "metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": B.world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": head["ms_per_step"], "higher_is_better": True,
            "scaling": "weak" if args.shard == "replicas" else "strong", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic", "config": head["config"], "clocks": head["clocks"], "e2e": head["e2e"],
            "gpu_launches": head["gpu_launches"], "roofline": head["roofline"],
            "wall_s_timed_region": head["wall_s_timed_region"],
        }
        out["config"]["headline"] = ("BASELINE.json's metric names no config; the headline is the largest single-GPU config "
                                     f"({HEADLINE}) unless --workload says otherwise; every other config is printed as its own "
                                     "{\"per_config\": ...} line before this one and summarised in all_configs")
        if "shard_check" in head:
            out["shard_check"] = head["shard_check"]
        if "cpu_baseline" in head:
            out["cpu_baseline"] = head["cpu_baseline"]
        per_all = {args.workload: head}
        per_all.update(per)

        def brief(r):
            rf, e, c = r["roofline"], r.get("e2e") or {}, r.get("cpu_baseline") or {}
            b = {"ms_per_step": round(r["ms_per_step"], 4), "steps": r["steps"], "warmup": r["warmup"], "value": float(f"{r['value']:.4g}"),
                 "e2e_ms_per_step": round(e["ms_per_step"], 4) if e else None, "e2e_value": float(f"{e['value']:.4g}") if e else None,
                 "segments_per_step": r["config"]["segments_per_step"], "gpu_launches": r["gpu_launches"],
                 "bound": rf["bound"], "roofline_frac": round(rf["frac"], 4) if rf.get("frac") is not None else None,
                 "march_ms_per_launch": round(rf["kernel_ms_per_launch"], 4), "march_share": round(rf["kernel_share_of_step"] or 0.0, 4),
                 "dram_frac": round(rf["dram_frac"], 4) if rf.get("dram_frac") is not None else None,
                 "sm_mhz": r["clocks"].get("sm_mhz"), "reasons": r["clocks"].get("reasons"),
                 "device_bytes_high_water": r["config"]["library_device_bytes_high_water"]}
            if c:
                b["cpu_oracle_value"] = float(f"{c['value']:.4g}")
            return b

        out["config"]["all_configs"] = {k: brief(per_all[k]) for k in sorted(per_all)}
        for k in sorted(per):          # the other configs in full, one line each, before the headline line
            line = {"per_config": k}
            line.update({kk: vv for kk, vv in per[k].items() if kk != "wall_s_timed_region"})
            print(json.dumps(line))
        if "alt_single_direction" in head:
            out["alt_single_direction"] = head["alt_single_direction"]
        print(json.dumps(out))
    if B.world > 1:
        B.dist.barrier()
        B.dist.destroy_process_group()


if __name__ == "__main__":
    main()
