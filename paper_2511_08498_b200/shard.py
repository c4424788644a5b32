"""Multi-GPU plumbing: how the path shards over ranks.

Rays are independent ("long characteristics is an embarrassingly parallel algorithm") and the rows of J
are disjoint per probe, so the path needs no exchange step.  Two ways to use N ranks, both one process per GPU:

  * "atmospheres" (bench.py default, weak scaling): every rank solves its own seeded atmosphere; torch.distributed is
    used only for the barrier and for the max-over-ranks of the device time / the sum of the emitted segments.
  * "probes": one atmosphere replicated on every rank, the probe list cut into contiguous, warp-aligned ranges; the
    only collective is one all-gather of the J rows at the end.

Nothing of the method's arithmetic lives here.
"""
from __future__ import annotations

from typing import Tuple

import torch
import torch.distributed as dist


def rank_seed(base_seed: int, rank: int) -> int:
    """Seed of rank `rank`'s own atmosphere in the weak-scaling run."""
    return int(base_seed) + 1000 * int(rank)


def probe_range(n_probes: int, world: int, rank: int, align: int = 32) -> Tuple[int, int]:
    """Contiguous [lo, hi) slice of the probe list owned by `rank`.  Cuts fall on multiples of `align` (a warp of
    probes) so that no warp straddles two ranks; the ranges tile [0, n_probes) exactly and differ by less than two warps."""
    if world <= 0 or not (0 <= rank < world):
        raise ValueError("rank outside the world")
    n_units = (n_probes + align - 1) // align
    base, extra = divmod(n_units, world)
    lo_u = rank * base + min(rank, extra)
    hi_u = lo_u + base + (1 if rank < extra else 0)
    return min(n_probes, lo_u * align), min(n_probes, hi_u * align)


def job_totals(device_ms: float, units: float, device="cpu") -> Tuple[float, float]:
    """(max over ranks of the device time, sum over ranks of the units processed).  One rank: the inputs."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(device_ms), float(units)
    t = torch.tensor([float(device_ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def gather_J(J_local: torch.Tensor, n_probes: int, align: int = 32) -> torch.Tensor:
    """All-gather of the per-rank J rows ("probes" mode) into the full [n_probes][n_lambda] array on every rank.
    Ranges may differ in length, so every rank pads to the longest before the collective."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return J_local
    world = dist.get_world_size()
    spans = [probe_range(n_probes, world, r, align) for r in range(world)]
    longest = max(hi - lo for lo, hi in spans)
    pad = torch.zeros((longest, J_local.shape[1]), dtype=J_local.dtype, device=J_local.device)
    pad[: J_local.shape[0]] = J_local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad)
    return torch.cat([parts[r][: hi - lo] for r, (lo, hi) in enumerate(spans)], dim=0)
