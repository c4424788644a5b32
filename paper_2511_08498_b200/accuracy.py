"""VLM accuracy report (BASELINE.json north_star: "the accuracy of VLM against the exact full-resolution
march is reported separately as the 99.9th-percentile relative error in J").

Both sides run on the GPU through the C ABI: the approximate side is the workload's own variant and level
table (VLM + HDDA); the exact side is the same library at level 0 -- `max_level = 0` for the isotropic
variant, `DEX_CLASSIC` (per-voxel velocity, brute-force line profile in every cell and direction; the
paper's ground truth) for the anisotropic ones.  The level-0 / Classic march is itself
parity-checked against the oracle in tests/test_gpu_parity.py.  The paper's Table 3 quotes the same
percentiles for level populations; J is what this hot path produces.

  python -m paper_2511_08498_b200.accuracy --workload C2 [--n-probes N] [--metric relvar|iod_log] [--caps paper]

Prints one JSON line: percentiles of |J_vlm - J_exact| / J_exact over (probe, wavelength), the level
histogram per batch (Table-2 style), segment counts and march times of both sides.
Reported, not gated.
"""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def level_histogram(levels: np.ndarray, max_level: int) -> list:
    """[n_batch][max_level + 2] brick counts for levels -1, 0, ..., max_level."""
    return [[int((row == m).sum()) for m in range(-1, max_level + 1)] for row in levels]


def percentiles(rel: np.ndarray) -> dict:
    qs = (50.0, 90.0, 99.0, 99.9)
    out = {f"p{q:g}": float(np.percentile(rel, q)) for q in qs}
    out["max"] = float(rel.max()) if rel.size else 0.0
    return out


PAPER_CAPS = (6.0, 24.0, 96.0, 384.0)   # level <= 0, 1, 2, 3 below these distances (voxels): PAPER.md:347-349, T8


def run(workload: str, n=None, n_dirs=None, n_probes=None, metric=None, thr=None, gate=None, max_level=None,
        caps=None, device="cuda:0", single_direction=False) -> dict:
    import torch
    from . import binding as B
    from . import pipeline
    from workloads import make

    wl = make(workload, n=n, n_dirs=n_dirs, n_probes=n_probes)
    if metric is not None:
        wl.metric = {"iod_log": 0, "relvar": 1}[metric]
    if thr is not None:
        wl.thr_eta = wl.thr_chi = float(thr)
    if gate is not None:
        wl.tau_gate = float(gate)
    if max_level is not None:
        wl.max_level = int(max_level)
    dw = pipeline.upload(wl, device, non_blocking=False)
    grid = pipeline.build_grid(dw)
    stream = torch.cuda.current_stream()

    def solve(use_caps=False, **override):
        mips = pipeline.build_mips(dw, grid, **override)
        if use_caps and caps:
            mips.set_level_caps(caps)
        seg = torch.zeros(1, dtype=torch.int64, device=device)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        J = pipeline.mean_intensity(dw, grid, mips, segment_count=seg)
        b.record(stream)
        torch.cuda.synchronize()
        lv = mips.levels()
        mips.destroy()
        return J.cpu().numpy().astype(np.float64), int(seg.item()), a.elapsed_time(b), lv

    def solve_single_direction():
        # PAPER.md:396 / DESIGN.md T11: per-direction Classic fields -> ISO VLM -> one-direction march, accumulated
        seg = torch.zeros(1, dtype=torch.int64, device=device)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        pipeline.mean_intensity_single_direction(dw, grid, level_caps=caps)        # warm the pool
        a.record(stream)
        J, lvs = pipeline.mean_intensity_single_direction(dw, grid, level_caps=caps, segment_count=seg, want_levels=True)
        b.record(stream)
        torch.cuda.synchronize()
        return J.cpu().numpy().astype(np.float64), int(seg.item()), a.elapsed_time(b), lvs

    sd = None
    if single_direction:
        if wl.variant == B.DEX_ISO:
            raise SystemExit("--single-direction needs an anisotropic workload (C3, C4, C5)")
        J_sd, seg_sd, ms_sd, lv_sd = solve_single_direction()
        sd = (J_sd, seg_sd, ms_sd, lv_sd)
    J_vlm, seg_vlm, ms_vlm, lv = solve(use_caps=True)
    if wl.variant == B.DEX_ISO:
        J_ex, seg_ex, ms_ex, _ = solve(max_level=0)
        exact = "same variant at max_level 0"
    else:
        J_ex, seg_ex, ms_ex, _ = solve(variant=B.DEX_CLASSIC, max_level=0)
        exact = "DEX_CLASSIC (per-voxel velocity, level 0; PAPER.md:365)"
    grid.destroy()
    lit = J_ex > 0.0                       # probes/wavelengths that see no emitting cell have J = 0 on both sides
    rel = np.abs(J_vlm[lit] - J_ex[lit]) / J_ex[lit]
    assert (J_vlm[~lit] == 0.0).all()
    hist = np.asarray(level_histogram(lv, wl.max_level))
    extra = {}
    if sd is not None:
        J_sd, seg_sd, ms_sd, lv_sd = sd
        h_sd = np.asarray(level_histogram(lv_sd.reshape(-1, lv_sd.shape[-1]), wl.max_level))
        extra["single_direction"] = {
            "what": "dex_mean_intensity_single_direction: per direction Classic fields -> ISO VLM -> march (PAPER.md:396); "
                    "ms covers fields + mips builds + marches of all directions",
            "rel_err_J": percentiles(np.abs(J_sd[lit] - J_ex[lit]) / J_ex[lit]), "segments": seg_sd, "ms_total": ms_sd,
            "level_histogram_mean_fraction": (h_sd.mean(axis=0) / h_sd[0].sum()).round(4).tolist(),
        }
    return {
        **extra,
        "report": "vlm_accuracy_J", "workload": wl.name, "dims": list(wl.dims[:wl.ndim]), "variant": int(wl.variant),
        "metric": "relvar" if wl.metric == 1 else "iod_log", "thr": float(wl.thr_eta), "tau_gate": float(wl.tau_gate),
        "max_level": int(wl.max_level), "level_cap_t": list(caps) if caps else [], "n_probes": int(wl.probe_pos.shape[0]), "n_dirs": int(wl.dirs.shape[0]),
        "n_lambda": int(wl.n_lambda), "exact_side": exact, "rel_err_J": percentiles(rel),
        "values_compared": int(rel.size), "segments_vlm": seg_vlm, "segments_exact": seg_ex,
        "segment_ratio": seg_ex / max(1, seg_vlm), "march_ms_vlm": ms_vlm, "march_ms_exact": ms_ex,
        "level_histogram_levels": list(range(-1, wl.max_level + 1)),
        "level_histogram_mean_fraction": (hist.mean(axis=0) / hist[0].sum()).round(4).tolist(),
        "level_histogram_per_batch": hist.tolist(),
    }


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="C2", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--n", type=int, default=None)
    ap.add_argument("--n-dirs", type=int, default=None)
    ap.add_argument("--n-probes", type=int, default=None)
    ap.add_argument("--metric", default=None, choices=["relvar", "iod_log"])
    ap.add_argument("--thr", type=float, default=None)
    ap.add_argument("--gate", type=float, default=None)
    ap.add_argument("--max-level", type=int, default=None)
    ap.add_argument("--caps", default=None,
                    help="near-field MIP cap thresholds: 'paper' (6,24,96,384 voxels) or a comma separated list")
    ap.add_argument("--single-direction", action="store_true",
                    help="also solve with per-direction VLM (dex_mean_intensity_single_direction) and report it")
    a = ap.parse_args()
    caps = None
    if a.caps:
        caps = PAPER_CAPS if a.caps == "paper" else tuple(float(v) for v in a.caps.split(","))
    print(json.dumps(run(a.workload, a.n, a.n_dirs, a.n_probes, a.metric, a.thr, a.gate, a.max_level, caps,
                         single_direction=a.single_direction)))


if __name__ == "__main__":
    main()
