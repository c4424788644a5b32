"""Host <-> device plumbing around the C-ABI calls (no arithmetic of the method lives here).

A `workload` is any object with the attributes of workloads.gen.Workload (numpy arrays on the host).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np
import torch

from . import binding as B

_SPEC_FIELDS = ("eta", "chi", "eta_bg", "chi_bg", "vel", "eta_star0", "chi_star0", "a0", "inv_dlamD", "lam")
_RAY_FIELDS = ("probe_pos", "dirs", "weights", "i0", "sin_incl")


@dataclass
class DeviceWorkload:
    wl: object
    t: dict = field(default_factory=dict)      # name -> device tensor
    h2d_bytes: int = 0


def pin(wl) -> dict:
    """Pinned host copies of every array the device needs (for the end-to-end timing leg)."""
    out = {}
    for name in _SPEC_FIELDS + _RAY_FIELDS + ("active",):
        a = getattr(wl, name, None)
        if a is None:
            continue
        t = torch.from_numpy(np.ascontiguousarray(a))
        out[name] = t.pin_memory() if torch.cuda.is_available() else t
    return out


def upload(wl, device="cuda:0", pinned: Optional[dict] = None, non_blocking=True) -> DeviceWorkload:
    dw = DeviceWorkload(wl=wl)
    src = pinned if pinned is not None else {n: torch.from_numpy(np.ascontiguousarray(getattr(wl, n)))
                                             for n in _SPEC_FIELDS + _RAY_FIELDS + ("active",)
                                             if getattr(wl, n, None) is not None}
    for name, t in src.items():
        dw.t[name] = t.to(device, non_blocking=non_blocking)
        dw.h2d_bytes += t.numel() * t.element_size()
    return dw


def build_grid(dw: DeviceWorkload, stream=None) -> B.Grid:
    wl = dw.wl
    return B.dex_build_sparse_grid(wl.ndim, wl.dims[:wl.ndim], wl.brick, wl.voxel_size, dw.t.get("active"), stream)


def build_mips(dw: DeviceWorkload, grid: B.Grid, stream=None, **override) -> B.Mips:
    wl = dw.wl
    g = lambda k: override.get(k, getattr(wl, k))
    t = dw.t
    return B.dex_build_vlm_mips(
        grid, g("variant"), wl.n_lambda, wl.lambda_batch, g("max_level"), g("metric"), g("thr_eta"), g("thr_chi"),
        g("tau_gate"), eta=t.get("eta"), chi=t.get("chi"), lam=t.get("lam"), eta_bg=t.get("eta_bg"),
        chi_bg=t.get("chi_bg"), vel=t.get("vel"), lambda0=wl.lambda0, eta_star0=t.get("eta_star0"),
        chi_star0=t.get("chi_star0"), a0=t.get("a0"), inv_dlamD=t.get("inv_dlamD"), active_lines=wl.active_lines,
        n_vbins=g("n_vbins"), c_light=wl.c_light, stream=stream)


def rays(dw: DeviceWorkload) -> B.Rays:
    t = dw.t
    return B.Rays(t["probe_pos"], t["dirs"], t.get("weights"), t.get("i0"), t.get("sin_incl"),
                  getattr(dw.wl, "interval", None))


def mean_intensity(dw: DeviceWorkload, grid: B.Grid, mips: B.Mips, J: Optional[torch.Tensor] = None,
                   segment_count: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    r = rays(dw)
    if J is None:
        J = torch.empty((r.n_probes, dw.wl.n_lambda), dtype=torch.float32, device=r.probe_pos.device)
    B.dex_mean_intensity(grid, mips, r, J, None, segment_count, stream)
    return J


def _mips_args(wl, t: dict, **override) -> dict:
    g = lambda k: override.get(k, getattr(wl, k))
    return dict(variant=g("variant"), n_lambda=wl.n_lambda, lambda_batch=wl.lambda_batch, max_level=g("max_level"),
                metric=g("metric"), thr_eta=g("thr_eta"), thr_chi=g("thr_chi"), tau_gate=g("tau_gate"), eta=t.get("eta"),
                chi=t.get("chi"), lam=t.get("lam"), eta_bg=t.get("eta_bg"), chi_bg=t.get("chi_bg"), vel=t.get("vel"),
                lambda0=wl.lambda0, eta_star0=t.get("eta_star0"), chi_star0=t.get("chi_star0"), a0=t.get("a0"),
                inv_dlamD=t.get("inv_dlamD"), active_lines=wl.active_lines, n_vbins=g("n_vbins"), c_light=wl.c_light)


def mean_intensity_pipelined(dw: DeviceWorkload, grid: B.Grid, batches_per_stage: int = 1, J: Optional[torch.Tensor] = None,
                             level_caps=None, segment_count: Optional[torch.Tensor] = None, want_levels=False,
                             stream=None, **override):
    """Per-iteration rebuild pipeline (include/dex.h dex_mean_intensity_pipelined): mips of stage s+1 are built while
    stage s is marched; returns (J, level table or None)."""
    r = rays(dw)
    if J is None:
        J = torch.empty((r.n_probes, dw.wl.n_lambda), dtype=torch.float32, device=r.probe_pos.device)
    lv = B.dex_mean_intensity_pipelined(grid, _mips_args(dw.wl, dw.t, **override), r, J, batches_per_stage, level_caps,
                                        segment_count, want_levels, stream)
    return J, lv


def direction_fields(dw: DeviceWorkload, grid: B.Grid, k: int, stream=None):
    """Classic eta, chi of the workload's anisotropic medium along quadrature direction k (dense device tensors)."""
    wl, t = dw.wl, dw.t
    dev = t["probe_pos"].device
    eta = torch.empty((wl.nvox, wl.n_lambda), dtype=torch.float32, device=dev)
    chi = torch.empty_like(eta)
    si = t.get("sin_incl")
    B.dex_direction_fields(grid, _mips_args(wl, t), t["dirs"][k], eta, chi, None if si is None else si[k:k + 1], stream)
    return eta, chi


def mean_intensity_single_direction(dw: DeviceWorkload, grid: B.Grid, J: Optional[torch.Tensor] = None, level_caps=None,
                                    segment_count: Optional[torch.Tensor] = None, want_levels=False, stream=None,
                                    **override):
    """Single-direction VLM (include/dex.h dex_mean_intensity_single_direction); returns (J, level tables or None)."""
    r = rays(dw)
    if J is None:
        J = torch.empty((r.n_probes, dw.wl.n_lambda), dtype=torch.float32, device=r.probe_pos.device)
    lv = B.dex_mean_intensity_single_direction(grid, _mips_args(dw.wl, dw.t, **override), r, J, level_caps,
                                               segment_count, want_levels, stream)
    return J, lv


def formal_solution(dw: DeviceWorkload, grid: B.Grid, mips: B.Mips, capture_batch: Optional[int] = None,
                    segment_count: Optional[torch.Tensor] = None, want_I=True, room: Optional[int] = None, stream=None):
    r = rays(dw)
    dev = r.probe_pos.device
    I = torch.empty((r.n_probes, r.n_dirs, dw.wl.n_lambda), dtype=torch.float32, device=dev) if want_I else None
    cap = None
    if capture_batch is not None:
        room = room if room is not None else int(sum(dw.wl.dims[:dw.wl.ndim])) + 16
        cap = B.VisitCapture(r.n_probes * r.n_dirs, room, capture_batch, dev)
    B.dex_formal_solution(grid, mips, r, I, cap, segment_count, stream)
    return I, cap


def solve_J_from_host(wl, device="cuda:0", pinned: Optional[dict] = None, J_host: Optional[torch.Tensor] = None):
    """The end-to-end call a user makes with HOST buffers: one dex_mean_intensity_host call (include/dex.h), which
    uploads the inputs, builds grid + mips, runs the fused march to J and copies J and the emitted-segment count
    back.  `pinned` = pin(wl) makes the copies asynchronous.  Returns (J numpy, segments, h2d_bytes, d2h_bytes)."""
    src = pinned if pinned is not None else {n: torch.from_numpy(np.ascontiguousarray(getattr(wl, n)))
                                             for n in _SPEC_FIELDS + _RAY_FIELDS + ("active",)
                                             if getattr(wl, n, None) is not None}
    r = B.Rays(src["probe_pos"], src["dirs"], src.get("weights"), src.get("i0"), src.get("sin_incl"),
               getattr(wl, "interval", None))
    if J_host is None:
        J_host = torch.empty((r.n_probes, wl.n_lambda), dtype=torch.float32)
        if torch.cuda.is_available():
            J_host = J_host.pin_memory()
    args = dict(variant=wl.variant, n_lambda=wl.n_lambda, lambda_batch=wl.lambda_batch, max_level=wl.max_level,
                metric=wl.metric, thr_eta=wl.thr_eta, thr_chi=wl.thr_chi, tau_gate=wl.tau_gate, eta=src.get("eta"),
                chi=src.get("chi"), lam=src.get("lam"), eta_bg=src.get("eta_bg"), chi_bg=src.get("chi_bg"),
                vel=src.get("vel"), lambda0=wl.lambda0, eta_star0=src.get("eta_star0"), chi_star0=src.get("chi_star0"),
                a0=src.get("a0"), inv_dlamD=src.get("inv_dlamD"), active_lines=wl.active_lines, n_vbins=wl.n_vbins,
                c_light=wl.c_light)
    with torch.cuda.device(device):
        nseg, h2d, d2h = B.dex_mean_intensity_host(wl.ndim, wl.dims[:wl.ndim], wl.brick, wl.voxel_size, src.get("active"),
                                                   args, r, J_host)
    return J_host.numpy(), nseg, h2d, d2h
