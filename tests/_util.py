"""Small helpers for the tests: hand-built workloads and independent geometry."""
from __future__ import annotations

import numpy as np

from workloads.gen import Workload, VARIANT_ISO, METRIC_RELVAR


def iso_workload(dims, brick, eta, chi, probes, dirs, active=None, weights=None, max_level=0,
                 metric=METRIC_RELVAR, thr=0.0, tau_gate=-1.0, h=1.0, W=None, i0=None, name="tiny"):
    """eta/chi: arrays of shape (.., Ny, Nx, n_lambda) or (.., Ny, Nx) (then n_lambda = 1 -> padded to W)."""
    ndim = len(dims)
    d3 = tuple(dims) + (1,) * (3 - ndim)
    eta = np.asarray(eta, dtype=np.float64)
    chi = np.asarray(chi, dtype=np.float64)
    if eta.ndim == ndim:
        eta = eta[..., None]
        chi = chi[..., None]
    nl = eta.shape[-1]
    if W is None:
        W = 8
    if nl % W:
        rep = W - nl % W
        eta = np.concatenate([eta] + [eta[..., -1:]] * rep, axis=-1)
        chi = np.concatenate([chi] + [chi[..., -1:]] * rep, axis=-1)
        if i0 is not None and np.asarray(i0).shape[-1] == nl:
            i0 = np.concatenate([i0] + [i0[..., -1:]] * rep, axis=-1)
        nl = eta.shape[-1]
    nvox = int(np.prod(d3))
    if active is None:
        active = np.ones(nvox, dtype=np.uint8)
    dirs = np.ascontiguousarray(np.asarray(dirs, dtype=np.float32).reshape(-1, ndim))
    if weights is None:
        weights = np.full(dirs.shape[0], 1.0 / dirs.shape[0], dtype=np.float32)
    return Workload(
        name=name, ndim=ndim, dims=d3, brick=brick, voxel_size=h,
        active=np.ascontiguousarray(np.asarray(active, dtype=np.uint8).ravel()),
        variant=VARIANT_ISO, n_lambda=nl, lambda_batch=W, max_level=max_level, metric=metric,
        thr_eta=thr, thr_chi=thr, tau_gate=tau_gate,
        probe_pos=np.ascontiguousarray(np.asarray(probes, dtype=np.float32).reshape(-1, ndim)),
        dirs=dirs, weights=np.asarray(weights, dtype=np.float32),
        i0=None if i0 is None else np.ascontiguousarray(np.asarray(i0, dtype=np.float32)),
        eta=np.ascontiguousarray(eta.reshape(nvox, nl).astype(np.float32)),
        chi=np.ascontiguousarray(chi.reshape(nvox, nl).astype(np.float32)),
    )


def path_to_boundary(probe, omega, dims):
    """fp64 length of the upwind characteristic x(s) = p - s w from the probe to the box boundary."""
    o = np.asarray(probe, dtype=np.float32).astype(np.float64)
    d = -np.asarray(omega, dtype=np.float32).astype(np.float64)
    t = np.inf
    for a in range(len(o)):
        if d[a] > 0:
            t = min(t, (dims[a] - o[a]) / d[a])
        elif d[a] < 0:
            t = min(t, (0.0 - o[a]) / d[a])
    return t


def unit_dirs_2d(angles):
    a = np.asarray(angles, dtype=np.float64)
    return np.stack([np.cos(a), np.sin(a)], axis=1).astype(np.float32)


def random_unit_dirs(n, ndim, rng):
    v = rng.standard_normal((n, ndim))
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    return v.astype(np.float32)


def fig5_levels():
    """PAPER.md:148 / Fig. 5: 32x32 model, 4x4 blocks of 8x8; blocks 0,1,2,4,8,12,15 empty, block 9
    refined to 4x4 (level 1), block 10 to 2x2 (level 2), all others fully refined (level 0)."""
    lv = np.zeros(16, dtype=np.int8)
    for b in (0, 1, 2, 4, 8, 12, 15):
        lv[b] = -1
    lv[9] = 1
    lv[10] = 2
    return lv


def max_rel(a, b):
    """Intensity comparison rule: |a-b|/|b|, both exactly 0 counts as 0."""
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    den = np.abs(b)
    diff = np.abs(a - b)
    with np.errstate(all="ignore"):
        r = np.where(diff == 0.0, 0.0, diff / den)
    return float(np.max(r)) if r.size else 0.0
