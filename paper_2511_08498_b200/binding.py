"""Thin ctypes binding of libdex.so (include/dex.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; torch is used for device
memory and streams.  There is no CPU fallback: if the shared library is missing, importing this
module raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdex.so")

DEX_OK, DEX_ERR_INVALID_ARG, DEX_ERR_SHAPE, DEX_ERR_UNSUPPORTED, DEX_ERR_OOM, DEX_ERR_CUDA, DEX_ERR_CAPACITY = range(7)
DEX_ISO, DEX_VELINTERP, DEX_CAV, DEX_CLASSIC = range(4)
DEX_METRIC_IOD_LOG, DEX_METRIC_RELVAR = 0, 1
DEX_CHAIN_ETA, DEX_CHAIN_CHI, DEX_CHAIN_VEL, DEX_CHAIN_LINE, DEX_CHAIN_VTAB = range(5)
DEX_MAX_LINES = 4
_STATUS = {0: "DEX_OK", 1: "DEX_ERR_INVALID_ARG", 2: "DEX_ERR_SHAPE", 3: "DEX_ERR_UNSUPPORTED", 4: "DEX_ERR_OOM",
           5: "DEX_ERR_CUDA", 6: "DEX_ERR_CAPACITY"}

EXPORTS = (
    "dex_last_error", "dex_version", "dex_build_sparse_grid", "dex_grid_info", "dex_grid_get_slots",
    "dex_destroy_grid", "dex_build_vlm_mips", "dex_mips_get_levels", "dex_mips_set_levels", "dex_mips_set_level_caps", "dex_mips_velocity_bin_report",
    "dex_mips_get_packed_levels", "dex_mips_get_level_data", "dex_destroy_mips", "dex_formal_solution",
    "dex_mean_intensity", "dex_mean_intensity_host", "dex_mean_intensity_pipelined", "dex_pool_high_water", "dex_trim", "dex_direction_fields",
    "dex_mean_intensity_single_direction", "dex_voigt_profile", "dex_launch_count", "dex_march_timing_enable", "dex_march_timing_read", "dex_march_work_read",
    "dex_set_lanes_per_ray", "dex_get_lanes_per_ray", "dex_measure_fp32_peak", "dex_set_tuning",
    "dex_brick_slots_static", "dex_last_march_mapping",
)
DEX_STATIC_MAX_BRICKS = 1 << 20


class DexError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


class _GridDesc(C.Structure):
    _fields_ = [("ndim", C.c_int), ("dims", C.c_int * 3), ("brick", C.c_int), ("voxel_size", C.c_float)]


class _MipsDesc(C.Structure):
    _fields_ = [
        ("variant", C.c_int), ("n_lambda", C.c_int), ("lambda_batch", C.c_int), ("max_level", C.c_int),
        ("metric", C.c_int), ("thr_eta", C.c_float), ("thr_chi", C.c_float), ("tau_gate", C.c_float),
        ("d_lambda", C.c_void_p), ("d_eta", C.c_void_p), ("d_chi", C.c_void_p), ("d_eta_bg", C.c_void_p),
        ("d_chi_bg", C.c_void_p), ("d_vel", C.c_void_p), ("n_lines", C.c_int), ("h_lambda0", C.c_void_p),
        ("d_eta_star0", C.c_void_p), ("d_chi_star0", C.c_void_p), ("d_a0", C.c_void_p), ("d_inv_dlamD", C.c_void_p),
        ("h_active_lines", C.c_void_p), ("n_vbins", C.c_int), ("c_light", C.c_float),
        ("lambda_stride", C.c_int),
    ]


class _Rays(C.Structure):
    _fields_ = [("n_probes", C.c_int64), ("d_probe_pos", C.c_void_p), ("n_dirs", C.c_int), ("d_dirs", C.c_void_p),
                ("d_weights", C.c_void_p), ("d_i0", C.c_void_p), ("d_sin_incl", C.c_void_p),
                ("t_begin", C.c_float), ("t_end", C.c_float), ("accumulate", C.c_int)]


class _Capture(C.Structure):
    _fields_ = [("d_counts", C.c_void_p), ("d_records", C.c_void_p), ("d_ds", C.c_void_p), ("capacity", C.c_int64),
                ("d_offsets", C.c_void_p), ("batch", C.c_int)]


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    L.dex_last_error.restype = C.c_char_p
    L.dex_version.restype = C.c_char_p
    L.dex_launch_count.restype = C.c_int64
    L.dex_build_sparse_grid.argtypes = [C.POINTER(_GridDesc), C.c_void_p, C.c_void_p, C.POINTER(C.c_void_p)]
    L.dex_brick_slots_static.argtypes = [C.POINTER(_GridDesc), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    L.dex_grid_info.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    L.dex_grid_get_slots.argtypes = [C.c_void_p, C.c_void_p]
    L.dex_destroy_grid.argtypes = [C.c_void_p]
    L.dex_destroy_grid.restype = None
    L.dex_build_vlm_mips.argtypes = [C.c_void_p, C.POINTER(_MipsDesc), C.c_void_p, C.POINTER(C.c_void_p)]
    L.dex_mips_get_levels.argtypes = [C.c_void_p, C.c_void_p]
    L.dex_mips_set_levels.argtypes = [C.c_void_p, C.c_void_p]
    L.dex_mips_set_level_caps.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
    L.dex_mips_velocity_bin_report.argtypes = [C.c_void_p, C.c_float, C.c_void_p, C.c_void_p]
    L.dex_mips_get_packed_levels.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.POINTER(C.c_int64)]
    L.dex_mips_get_level_data.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p]
    L.dex_destroy_mips.argtypes = [C.c_void_p]
    L.dex_destroy_mips.restype = None
    L.dex_formal_solution.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(_Rays), C.c_void_p, C.POINTER(_Capture),
                                      C.c_void_p, C.c_void_p]
    L.dex_mean_intensity.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(_Rays), C.c_void_p, C.c_void_p, C.c_void_p,
                                     C.c_void_p]
    L.dex_mean_intensity_host.argtypes = [C.POINTER(_GridDesc), C.c_void_p, C.POINTER(_MipsDesc), C.POINTER(_Rays),
                                          C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.POINTER(C.c_int64),
                                          C.c_void_p]
    L.dex_mean_intensity_pipelined.argtypes = [C.c_void_p, C.POINTER(_MipsDesc), C.POINTER(_Rays), C.c_int, C.c_int,
                                               C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    L.dex_direction_fields.argtypes = [C.c_void_p, C.POINTER(_MipsDesc), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                       C.c_void_p]
    L.dex_mean_intensity_single_direction.argtypes = [C.c_void_p, C.POINTER(_MipsDesc), C.POINTER(_Rays), C.c_int,
                                                      C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    L.dex_pool_high_water.argtypes = [C.POINTER(C.c_int64), C.c_int]
    L.dex_voigt_profile.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_int, C.c_void_p]
    L.dex_march_timing_enable.argtypes = [C.c_int]
    L.dex_march_timing_enable.restype = None
    L.dex_march_timing_read.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_int64), C.c_int]
    L.dex_march_work_read.argtypes = [C.POINTER(C.c_int64), C.c_int]
    L.dex_set_lanes_per_ray.argtypes = [C.c_int]
    L.dex_set_tuning.argtypes = [C.c_char_p, C.c_int]
    L.dex_trim.argtypes = [C.POINTER(C.c_int64)]
    L.dex_get_lanes_per_ray.argtypes = [C.c_int64, C.c_int, C.c_int, C.POINTER(C.c_int)]
    L.dex_last_march_mapping.argtypes = [C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int)]
    L.dex_measure_fp32_peak.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_void_p]
    return L


_L = _load()


def _check(status):
    if status != DEX_OK:
        raise DexError(status, (_L.dex_last_error() or b"").decode())


def _ptr(t: Optional[torch.Tensor], dtype=None, cuda=True):
    if t is None:
        return None
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"expected {dtype}, got {t.dtype}")
    if cuda and not t.is_cuda:
        raise TypeError("expected a CUDA tensor")
    if not cuda and t.is_cuda:
        raise TypeError("expected a host tensor")
    if not t.is_contiguous():
        raise TypeError("expected a contiguous tensor")
    return t.data_ptr()


def _stream(stream):
    if stream is None:
        return torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else 0
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


def dex_version() -> str:
    return _L.dex_version().decode()


def dex_launch_count() -> int:
    return int(_L.dex_launch_count())


def dex_set_lanes_per_ray(lanes: int):
    _check(_L.dex_set_lanes_per_ray(int(lanes)))


def dex_trim() -> int:
    """Return the library pool's unused device memory to the driver; returns the bytes it still holds."""
    v = C.c_int64(0)
    _check(_L.dex_trim(C.byref(v)))
    return v.value


def dex_get_lanes_per_ray(n_probes: int, n_dirs: int, n_lambda: int = 1) -> int:
    """Predicted lanes per ray of a whole-spectrum fused-J march (see dex_last_march_mapping for what a march ran with)."""
    v = C.c_int(0)
    _check(_L.dex_get_lanes_per_ray(int(n_probes), int(n_dirs), int(n_lambda), C.byref(v)))
    return v.value


def dex_last_march_mapping() -> dict:
    """What the last march launched from this thread ran with: lanes per ray, directions per block of the direction split
    (0 = not split), wavelength batches per group of the memoised march (0 = not memoised)."""
    a, b, c = C.c_int(0), C.c_int(0), C.c_int(0)
    _check(_L.dex_last_march_mapping(C.byref(a), C.byref(b), C.byref(c)))
    return {"lanes_per_ray": a.value, "dirs_per_block": b.value, "memo_batches_per_group": c.value}


def dex_measure_fp32_peak(stream=None):
    """(TFLOP/s of scalar FFMA chains, TFLOP/s of packed FFMA2 chains), measured on the current device."""
    a, b = C.c_double(0), C.c_double(0)
    _check(_L.dex_measure_fp32_peak(C.byref(a), C.byref(b), _stream(stream)))
    return a.value, b.value


def dex_set_tuning(name: str, value: int):
    _check(_L.dex_set_tuning(name.encode(), int(value)))


def dex_march_timing_enable(on: bool):
    _L.dex_march_timing_enable(1 if on else 0)


def dex_march_timing_read(reset=True):
    ms, n = C.c_double(0), C.c_int64(0)
    _check(_L.dex_march_timing_read(C.byref(ms), C.byref(n), 1 if reset else 0))
    return ms.value, n.value


def dex_march_work_read(reset=True) -> int:
    v = C.c_int64(0)
    _check(_L.dex_march_work_read(C.byref(v), 1 if reset else 0))
    return v.value


class Grid:
    def __init__(self, handle, ndim, dims, brick, voxel_size):
        self.handle, self.ndim, self.dims, self.brick, self.voxel_size = handle, ndim, tuple(dims), brick, voxel_size

    def info(self):
        nb, na = C.c_int64(0), C.c_int64(0)
        _check(_L.dex_grid_info(self.handle, C.byref(nb), C.byref(na)))
        return nb.value, na.value

    def slots(self) -> np.ndarray:
        nb, _ = self.info()
        out = np.empty(nb, dtype=np.int32)
        _check(_L.dex_grid_get_slots(self.handle, out.ctypes.data))
        return out

    def destroy(self):
        if self.handle:
            _L.dex_destroy_grid(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def dex_build_sparse_grid(ndim, dims, brick, voxel_size, active: Optional[torch.Tensor] = None, stream=None) -> Grid:
    d = _GridDesc()
    d.ndim = ndim
    dd = list(dims) + [1] * (3 - len(dims))
    for a in range(3):
        d.dims[a] = int(dd[a])
    d.brick = int(brick)
    d.voxel_size = float(voxel_size)
    h = C.c_void_p()
    _check(_L.dex_build_sparse_grid(C.byref(d), _ptr(active, torch.uint8), _stream(stream), C.byref(h)))
    return Grid(h, ndim, dd, brick, voxel_size)


def dex_brick_slots_static(ndim, dims, brick, voxel_size, active: Optional[torch.Tensor], slot: torch.Tensor,
                           active_bricks: torch.Tensor, n_active: torch.Tensor, stream=None):
    """Step a1 for callers that cannot allocate on the device (a fixed memory budget, a host application that owns the
    allocator, a loop that cannot wait on the driver): brick slots, slot -> brick list and active count written into
    the caller's int32 CUDA tensors `slot` [n_bricks], `active_bricks` [n_bricks], `n_active` [1].  Nothing is
    allocated, nothing synchronises; the flag scratch is a 4 MiB array inside libdex.so, so at most
    DEX_STATIC_MAX_BRICKS bricks (DexError otherwise) and no two overlapping calls on one GPU.  See include/dex.h."""
    d = _GridDesc()
    d.ndim = ndim
    dd = list(dims) + [1] * (3 - len(dims))
    for a in range(3):
        d.dims[a] = int(dd[a])
    d.brick = int(brick)
    d.voxel_size = float(voxel_size)
    _check(_L.dex_brick_slots_static(C.byref(d), _ptr(active, torch.uint8), _ptr(slot, torch.int32),
                                     _ptr(active_bricks, torch.int32), _ptr(n_active, torch.int32), _stream(stream)))


class Mips:
    def __init__(self, handle, grid: Grid, n_lambda, lambda_batch, max_level, variant, n_lines=0, n_vbins=0, keep=()):
        self.handle, self.grid = handle, grid
        self.n_lambda, self.lambda_batch, self.max_level, self.variant = n_lambda, lambda_batch, max_level, variant
        self.n_lines, self.n_vbins = n_lines, n_vbins
        self.n_batch = n_lambda // lambda_batch
        self._keep = keep

    def levels(self) -> np.ndarray:
        nb, _ = self.grid.info()
        out = np.empty((self.n_batch, nb), dtype=np.int8)
        _check(_L.dex_mips_get_levels(self.handle, out.ctypes.data))
        return out

    def set_levels(self, levels: np.ndarray):
        lv = np.ascontiguousarray(levels, dtype=np.int8)
        nb, _ = self.grid.info()
        if lv.shape != (self.n_batch, nb):
            raise ValueError("levels must be [n_batch][n_bricks]")
        _check(_L.dex_mips_set_levels(self.handle, lv.ctypes.data))

    def set_level_caps(self, cap_t):
        """Near-field MIP cap thresholds (ascending distances in voxels; empty / None removes the cap)."""
        t = np.ascontiguousarray([] if cap_t is None else cap_t, dtype=np.float32)
        _check(_L.dex_mips_set_level_caps(self.handle, int(t.size), t.ctypes.data if t.size else None))

    def velocity_bin_report(self, factor: float = 2.0):
        """PAPER.md:200 diagnostic: (max spacing / thermal width per line, level-0 cells above `factor` per line)."""
        mx = np.zeros(max(1, self.n_lines), dtype=np.float32)
        over = np.zeros(max(1, self.n_lines), dtype=np.int64)
        _check(_L.dex_mips_velocity_bin_report(self.handle, float(factor), mx.ctypes.data, over.ctypes.data))
        return mx[:self.n_lines], over[:self.n_lines]

    def packed_levels(self, batch: int) -> np.ndarray:
        n = C.c_int64(0)
        _check(_L.dex_mips_get_packed_levels(self.handle, batch, None, C.byref(n)))
        out = np.empty(n.value, dtype=np.uint64)
        _check(_L.dex_mips_get_packed_levels(self.handle, batch, out.ctypes.data, C.byref(n)))
        return out

    def level_data(self, chain: int, level: int) -> np.ndarray:
        cells = 1
        shape = []
        for a in range(self.grid.ndim):
            shape.append(self.grid.dims[a] >> level)
        shape = shape[::-1]
        width = {DEX_CHAIN_ETA: (self.n_lambda,), DEX_CHAIN_CHI: (self.n_lambda,), DEX_CHAIN_VEL: (4,),
                 DEX_CHAIN_LINE: (self.n_lines, 4), DEX_CHAIN_VTAB: (self.n_vbins, self.n_lambda, 2)}[chain]
        out = np.empty(tuple(shape) + width, dtype=np.float32)
        _check(_L.dex_mips_get_level_data(self.handle, chain, level, out.ctypes.data))
        return out

    def destroy(self):
        if self.handle:
            _L.dex_destroy_mips(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def _mips_desc(variant, n_lambda, lambda_batch, max_level, metric, thr_eta, thr_chi, tau_gate, eta, chi, lam, eta_bg,
               chi_bg, vel, lambda0, eta_star0, chi_star0, a0, inv_dlamD, active_lines, n_vbins, c_light, cuda=True):
    """Fill a dex_mips_desc; returns (desc, n_lines, host arrays that must outlive the call)."""
    d = _MipsDesc()
    d.variant, d.n_lambda, d.lambda_batch, d.max_level, d.metric = int(variant), int(n_lambda), int(lambda_batch), int(max_level), int(metric)
    d.thr_eta, d.thr_chi, d.tau_gate = float(thr_eta), float(thr_chi), float(tau_gate)
    f32 = torch.float32
    d.d_lambda, d.d_eta, d.d_chi = _ptr(lam, f32, cuda), _ptr(eta, f32, cuda), _ptr(chi, f32, cuda)
    d.d_eta_bg, d.d_chi_bg, d.d_vel = _ptr(eta_bg, f32, cuda), _ptr(chi_bg, f32, cuda), _ptr(vel, f32, cuda)
    keep = []
    n_lines = 0
    if lambda0 is not None:
        l0 = np.ascontiguousarray(lambda0, dtype=np.float32)
        keep.append(l0)
        n_lines = l0.shape[0]
        d.h_lambda0 = l0.ctypes.data
    d.n_lines = n_lines
    d.d_eta_star0, d.d_chi_star0 = _ptr(eta_star0, f32, cuda), _ptr(chi_star0, f32, cuda)
    d.d_a0, d.d_inv_dlamD = _ptr(a0, f32, cuda), _ptr(inv_dlamD, f32, cuda)
    if active_lines is not None:
        al = np.ascontiguousarray(active_lines, dtype=np.int8)
        if al.shape != (n_lambda // lambda_batch, DEX_MAX_LINES):
            raise ValueError("active_lines must be [n_batch][4]")
        keep.append(al)
        d.h_active_lines = al.ctypes.data
    d.n_vbins = int(n_vbins)
    d.c_light = float(c_light)
    return d, n_lines, keep


def dex_build_vlm_mips(grid: Grid, variant, n_lambda, lambda_batch, max_level, metric, thr_eta, thr_chi, tau_gate,
                       eta=None, chi=None, lam=None, eta_bg=None, chi_bg=None, vel=None, lambda0=None,
                       eta_star0=None, chi_star0=None, a0=None, inv_dlamD=None, active_lines=None, n_vbins=0,
                       c_light=299792.458, stream=None) -> Mips:
    d, n_lines, keep = _mips_desc(variant, n_lambda, lambda_batch, max_level, metric, thr_eta, thr_chi, tau_gate, eta,
                                  chi, lam, eta_bg, chi_bg, vel, lambda0, eta_star0, chi_star0, a0, inv_dlamD,
                                  active_lines, n_vbins, c_light)
    h = C.c_void_p()
    _check(_L.dex_build_vlm_mips(grid.handle, C.byref(d), _stream(stream), C.byref(h)))
    del keep
    return Mips(h, grid, n_lambda, lambda_batch, 0 if variant == DEX_CLASSIC else max_level, variant, n_lines, int(n_vbins))


class Rays:
    def __init__(self, probe_pos: torch.Tensor, dirs: torch.Tensor, weights: Optional[torch.Tensor] = None,
                 i0: Optional[torch.Tensor] = None, sin_incl: Optional[torch.Tensor] = None, interval=None):
        self.probe_pos, self.dirs, self.weights, self.i0, self.sin_incl = probe_pos, dirs, weights, i0, sin_incl
        self.interval = interval            # (t_begin, t_end) in voxels from the probe, None = to the boundary
        self.n_probes, self.n_dirs = int(probe_pos.shape[0]), int(dirs.shape[0])

    def struct(self, cuda=True):
        r = _Rays()
        f32 = torch.float32
        r.n_probes, r.n_dirs = self.n_probes, self.n_dirs
        r.d_probe_pos, r.d_dirs = _ptr(self.probe_pos, f32, cuda), _ptr(self.dirs, f32, cuda)
        r.d_weights, r.d_i0 = _ptr(self.weights, f32, cuda), _ptr(self.i0, f32, cuda)
        r.d_sin_incl = _ptr(self.sin_incl, f32, cuda)
        if self.interval is not None:
            r.t_begin, r.t_end = float(self.interval[0]), float(self.interval[1])
        return r


class VisitCapture:
    """Caller-owned capture buffers (validation mode): `room` records per ray."""

    def __init__(self, n_rays: int, room: int, batch: int, device, with_ds=True):
        self.counts = torch.zeros(n_rays, dtype=torch.int64, device=device)
        self.records = torch.zeros(n_rays * room, dtype=torch.int64, device=device)
        self.ds = torch.zeros(n_rays * room, dtype=torch.float32, device=device) if with_ds else None
        self.offsets = (torch.arange(n_rays, dtype=torch.int64, device=device) * room).contiguous()
        self.room, self.batch, self.n_rays = room, batch, n_rays

    def struct(self):
        c = _Capture()
        c.d_counts, c.d_records = self.counts.data_ptr(), self.records.data_ptr()
        c.d_ds = self.ds.data_ptr() if self.ds is not None else None
        c.capacity = self.n_rays * self.room
        c.d_offsets = self.offsets.data_ptr()
        c.batch = self.batch
        return c


def dex_formal_solution(grid: Grid, mips: Mips, rays: Rays, I: Optional[torch.Tensor], capture: Optional[VisitCapture] = None,
                        segment_count: Optional[torch.Tensor] = None, stream=None):
    r = rays.struct()
    cap = capture.struct() if capture is not None else None
    _check(_L.dex_formal_solution(grid.handle, mips.handle, C.byref(r), _ptr(I, torch.float32),
                                  C.byref(cap) if cap is not None else None, _ptr(segment_count, torch.int64),
                                  _stream(stream)))


def dex_mean_intensity(grid: Grid, mips: Mips, rays: Rays, J: torch.Tensor, I: Optional[torch.Tensor] = None,
                       segment_count: Optional[torch.Tensor] = None, stream=None):
    r = rays.struct()
    _check(_L.dex_mean_intensity(grid.handle, mips.handle, C.byref(r), _ptr(I, torch.float32), _ptr(J, torch.float32),
                                 _ptr(segment_count, torch.int64), _stream(stream)))


def dex_mean_intensity_host(ndim, dims, brick, voxel_size, active: Optional[torch.Tensor], mips_args: dict,
                            rays: Rays, J: torch.Tensor, stream=None):
    """include/dex.h dex_mean_intensity_host: the whole hot path from HOST tensors (pinned or pageable) to a host J.
    `mips_args` holds dex_build_vlm_mips' keyword arguments with host tensors.  Returns (segments, h2d, d2h bytes)."""
    g = _GridDesc()
    g.ndim = ndim
    dd = list(dims) + [1] * (3 - len(dims))
    for a in range(3):
        g.dims[a] = int(dd[a])
    g.brick, g.voxel_size = int(brick), float(voxel_size)
    a = dict(eta=None, chi=None, lam=None, eta_bg=None, chi_bg=None, vel=None, lambda0=None, eta_star0=None,
             chi_star0=None, a0=None, inv_dlamD=None, active_lines=None, n_vbins=0, c_light=299792.458)
    a.update(mips_args)
    d, _, keep = _mips_desc(cuda=False, **a)
    r = rays.struct(cuda=False)
    if J.is_cuda or J.dtype != torch.float32 or not J.is_contiguous() or J.numel() != rays.n_probes * int(a["n_lambda"]):
        raise TypeError("J must be a contiguous host fp32 tensor [n_probes][n_lambda]")
    seg, h2d, d2h = C.c_int64(0), C.c_int64(0), C.c_int64(0)
    _check(_L.dex_mean_intensity_host(C.byref(g), _ptr(active, torch.uint8, False), C.byref(d), C.byref(r), J.data_ptr(),
                                      C.byref(seg), C.byref(h2d), C.byref(d2h), _stream(stream)))
    del keep
    return seg.value, h2d.value, d2h.value


def dex_mean_intensity_pipelined(grid: Grid, mips_args: dict, rays: Rays, J: torch.Tensor, batches_per_stage: int = 1,
                                 level_caps=None, segment_count: Optional[torch.Tensor] = None, want_levels=False,
                                 stream=None):
    """include/dex.h dex_mean_intensity_pipelined: per-stage rebuild of the mips overlapped with the previous stage's
    march.  `mips_args` holds dex_build_vlm_mips' keyword arguments (device tensors).  Returns the level table
    [n_batch][n_bricks] when `want_levels`, else None."""
    a = dict(eta=None, chi=None, lam=None, eta_bg=None, chi_bg=None, vel=None, lambda0=None, eta_star0=None,
             chi_star0=None, a0=None, inv_dlamD=None, active_lines=None, n_vbins=0, c_light=299792.458)
    a.update(mips_args)
    d, _, keep = _mips_desc(**a)
    r = rays.struct()
    t = np.ascontiguousarray([] if level_caps is None else level_caps, dtype=np.float32)
    lv = None
    if want_levels:
        nb, _ = grid.info()
        lv = np.empty((int(a["n_lambda"]) // int(a["lambda_batch"]), nb), dtype=np.int8)
    _check(_L.dex_mean_intensity_pipelined(grid.handle, C.byref(d), C.byref(r), int(batches_per_stage), int(t.size),
                                           t.ctypes.data if t.size else None, _ptr(J, torch.float32),
                                           _ptr(segment_count, torch.int64), lv.ctypes.data if lv is not None else None,
                                           _stream(stream)))
    del keep
    return lv


_MIPS_DEFAULTS = dict(eta=None, chi=None, lam=None, eta_bg=None, chi_bg=None, vel=None, lambda0=None, eta_star0=None,
                      chi_star0=None, a0=None, inv_dlamD=None, active_lines=None, n_vbins=0, c_light=299792.458)


def dex_direction_fields(grid: Grid, mips_args: dict, omega: torch.Tensor, eta: torch.Tensor, chi: torch.Tensor,
                         sin_incl: Optional[torch.Tensor] = None, stream=None):
    """include/dex.h dex_direction_fields: Classic eta, chi along the direction `omega` (device fp32 [ndim]) into the
    dense device tensors eta, chi [nvox][n_lambda]."""
    a = dict(_MIPS_DEFAULTS)
    a.update(mips_args)
    d, _, keep = _mips_desc(**a)
    _check(_L.dex_direction_fields(grid.handle, C.byref(d), _ptr(omega, torch.float32), _ptr(sin_incl, torch.float32),
                                   _ptr(eta, torch.float32), _ptr(chi, torch.float32), _stream(stream)))
    del keep


def dex_mean_intensity_single_direction(grid: Grid, mips_args: dict, rays: Rays, J: torch.Tensor, level_caps=None,
                                        segment_count: Optional[torch.Tensor] = None, want_levels=False, stream=None):
    """include/dex.h dex_mean_intensity_single_direction.  Returns the level tables [n_dirs][n_batch][n_bricks] when
    `want_levels`, else None."""
    a = dict(_MIPS_DEFAULTS)
    a.update(mips_args)
    d, _, keep = _mips_desc(**a)
    r = rays.struct()
    t = np.ascontiguousarray([] if level_caps is None else level_caps, dtype=np.float32)
    lv = None
    if want_levels:
        nb, _ = grid.info()
        lv = np.empty((rays.n_dirs, int(a["n_lambda"]) // int(a["lambda_batch"]), nb), dtype=np.int8)
    _check(_L.dex_mean_intensity_single_direction(grid.handle, C.byref(d), C.byref(r), int(t.size),
                                                  t.ctypes.data if t.size else None, _ptr(J, torch.float32),
                                                  _ptr(segment_count, torch.int64),
                                                  lv.ctypes.data if lv is not None else None, _stream(stream)))
    del keep
    return lv


def dex_pool_high_water(reset=False) -> int:
    v = C.c_int64(0)
    _check(_L.dex_pool_high_water(C.byref(v), int(bool(reset))))
    return v.value


def dex_voigt_profile(a: torch.Tensor, x: torch.Tensor, mode: int = 0, stream=None) -> torch.Tensor:
    """Validation: H(a, x) as the Core-and-Voigt march evaluates it (a fp32, x fp64 CUDA tensors of equal length)."""
    if a.numel() != x.numel():
        raise ValueError("a and x must have the same length")
    H = torch.empty(x.numel(), dtype=torch.float64, device=x.device)
    _check(_L.dex_voigt_profile(_ptr(a, torch.float32), _ptr(x, torch.float64), a.numel(), H.data_ptr(), int(mode),
                                _stream(stream)))
    return H
