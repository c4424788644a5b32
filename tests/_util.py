"""Small helpers for the tests: hand-built workloads and independent geometry."""
from __future__ import annotations

import numpy as np

from workloads.gen import Workload, VARIANT_ISO, METRIC_RELVAR, batch_workload  # noqa: F401


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


def crop_workload(wl, lo, size):
    """Sub-grid [lo, lo + size) (voxels, brick aligned, per axis x, y[, z]) of a workload with the same fields and
    build parameters and no rays.  Mips, cell tests and brick levels are brick-local, so building the crop must give
    exactly the full grid's result for these bricks: this is how the full-size builds are checked against the oracle
    without running the (slow, numpy) oracle build over the whole grid."""
    import copy
    nd = wl.ndim
    lo = tuple(int(v) for v in lo) + (0,) * (3 - nd)
    size = tuple(int(v) for v in size) + (1,) * (3 - nd)
    assert all(l % wl.brick == 0 and s % wl.brick == 0 for l, s in zip(lo[:nd], size[:nd]))
    nx, ny, nz = wl.dims
    sl = (slice(lo[2], lo[2] + size[2]), slice(lo[1], lo[1] + size[1]), slice(lo[0], lo[0] + size[0]))

    def per_voxel(a):            # [nvox][...]
        if a is None:
            return None
        g = a.reshape((nz, ny, nx) + a.shape[1:])[sl]
        return np.ascontiguousarray(g.reshape((-1,) + a.shape[1:]))

    def per_line(a):             # [n_lines][nvox]
        if a is None:
            return None
        g = a.reshape((a.shape[0], nz, ny, nx))[(slice(None),) + sl]
        return np.ascontiguousarray(g.reshape(a.shape[0], -1))

    out = copy.copy(wl)
    out.dims = size
    out.active = per_voxel(wl.active)
    for name in ("eta", "chi", "eta_bg", "chi_bg", "vel"):
        setattr(out, name, per_voxel(getattr(wl, name)))
    for name in ("eta_star0", "chi_star0", "a0", "inv_dlamD"):
        setattr(out, name, per_line(getattr(wl, name)))
    out.probe_pos = np.zeros((0, nd), dtype=np.float32)
    return out


def crop_brick_ids(wl, lo, size):
    """Brick indices (in the full grid's numbering) of the bricks of the crop, in the crop's own brick order."""
    nd, b = wl.ndim, wl.brick
    lo = tuple(int(v) for v in lo) + (0,) * (3 - nd)
    size = tuple(int(v) for v in size) + (b,) * (3 - nd)
    bd = wl.brick_dims
    ids = []
    for bz in range(lo[2] // b, lo[2] // b + (size[2] // b if nd == 3 else 1)):
        for by in range(lo[1] // b, (lo[1] + size[1]) // b):
            for bx in range(lo[0] // b, (lo[0] + size[0]) // b):
                ids.append((bz * bd[1] + by) * bd[0] + bx)
    return np.asarray(ids, dtype=np.int64)

