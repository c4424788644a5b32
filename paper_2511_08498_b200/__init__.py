"""B200-native long-characteristics formal solver (hot path of arxiv/paper_2511_08498).

Public surface: the four C-ABI calls of include/dex.h through their thin binding
(dex_build_sparse_grid, dex_build_vlm_mips, dex_formal_solution, dex_mean_intensity) plus the
`pipeline` helpers that move a workload's host arrays to the device and chain the calls.
Importing this package requires the compiled libdex.so (no CPU fallback).
"""
from .binding import (  # noqa: F401
    DEX_CAV, DEX_CHAIN_CHI, DEX_CHAIN_ETA, DEX_CHAIN_LINE, DEX_CHAIN_VEL, DEX_CHAIN_VTAB, DEX_CLASSIC, DEX_ISO,
    DEX_METRIC_IOD_LOG, DEX_METRIC_RELVAR, DEX_VELINTERP, DexError, Grid, Mips, Rays, VisitCapture,
    dex_build_sparse_grid, dex_build_vlm_mips, dex_formal_solution, dex_launch_count, dex_march_timing_enable,
    dex_march_timing_read, dex_march_work_read, dex_mean_intensity, dex_mean_intensity_host, dex_direction_fields, dex_mean_intensity_pipelined, dex_mean_intensity_single_direction, dex_pool_high_water, dex_trim, dex_set_lanes_per_ray, dex_get_lanes_per_ray, dex_measure_fp32_peak, dex_set_tuning, dex_version, dex_voigt_profile, dex_brick_slots_static, dex_last_march_mapping,
)
from . import pipeline, shard  # noqa: F401
