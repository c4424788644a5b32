"""Seeded input generators for configs C1..C5 (BASELINE.json `configs`).

The paper measures on a private prominence snapshot that is not
available; these synthetic atmospheres stand in for it and take its structure: smooth
regions punctuated by sharp interfaces, brick-granular sparsity
(PAPER.md:351), structure that differs per wavelength and many
orders of magnitude in opacity.

Everything here is *input construction*.  Nothing of the method (mip averaging, the
VLM test, traversal, line-profile evaluation, the formal solution) lives here.

Array conventions (shared by oracle and library):
  * voxel index  v = (z*Ny + y)*Nx + x   (x fastest), dims = (Nx, Ny, Nz)
  * per-voxel spectra are [nvox][n_lambda] fp32, lambda fastest
  * per-line fields are [n_lines][nvox] fp32
  * velocities are [nvox][ndim] fp32 in km/s, components (vx, vy[, vz])
  * probe positions [n_probes][ndim] fp32 in index space (voxel side = 1)
  * directions [n_dirs][ndim] fp32 are *propagation* directions (omega-hat, eq. 1)
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

C_LIGHT_KMS = 299792.458
CONFIG_NAMES = ("C1", "C2", "C3", "C4", "C5")
SEEDS = {"C1": 8498001, "C2": 8498002, "C3": 8498003, "C4": 8498004, "C5": 8498005}

VARIANT_ISO, VARIANT_VELINTERP, VARIANT_CAV, VARIANT_CLASSIC = 0, 1, 2, 3
METRIC_IOD_LOG, METRIC_RELVAR = 0, 1


@dataclass
class Workload:
    name: str
    ndim: int
    dims: tuple            # (Nx, Ny, Nz); Nz = 1 in 2D
    brick: int
    voxel_size: float
    active: np.ndarray     # uint8 [nvox]
    variant: int
    n_lambda: int
    lambda_batch: int
    max_level: int
    metric: int
    thr_eta: float
    thr_chi: float
    tau_gate: float
    # rays
    probe_pos: np.ndarray = None   # [n_probes][ndim] fp32
    dirs: np.ndarray = None        # [n_dirs][ndim] fp32
    weights: np.ndarray = None     # [n_dirs] fp32
    i0: Optional[np.ndarray] = None  # [n_dirs][n_lambda] fp32 or None (= 0)
    sin_incl: Optional[np.ndarray] = None  # [n_dirs] fp32 or None: 2.5D rays, sine of the inclination to the homogeneous axis
    interval: Optional[tuple] = None       # (t_begin, t_end) voxels from the probe: finite radiance interval, None = to the boundary
    # isotropic fields
    eta: Optional[np.ndarray] = None
    chi: Optional[np.ndarray] = None
    # anisotropic fields
    lam: Optional[np.ndarray] = None          # [n_lambda] fp32, nm
    eta_bg: Optional[np.ndarray] = None
    chi_bg: Optional[np.ndarray] = None
    vel: Optional[np.ndarray] = None          # [nvox][ndim] km/s
    n_lines: int = 0
    lambda0: Optional[np.ndarray] = None      # [n_lines] fp32
    eta_star0: Optional[np.ndarray] = None    # [n_lines][nvox]
    chi_star0: Optional[np.ndarray] = None
    a0: Optional[np.ndarray] = None
    inv_dlamD: Optional[np.ndarray] = None
    active_lines: Optional[np.ndarray] = None  # int8 [n_batch][4], -1 padded
    n_vbins: int = 0
    c_light: float = C_LIGHT_KMS
    notes: dict = field(default_factory=dict)

    @property
    def nvox(self) -> int:
        return int(self.dims[0]) * int(self.dims[1]) * int(self.dims[2])

    @property
    def n_batch(self) -> int:
        return self.n_lambda // self.lambda_batch

    @property
    def brick_dims(self) -> tuple:
        b = self.brick
        return (self.dims[0] // b, self.dims[1] // b, max(1, self.dims[2] // b) if self.ndim == 3 else 1)

    @property
    def n_bricks(self) -> int:
        bd = self.brick_dims
        return bd[0] * bd[1] * bd[2]


# --------------------------------------------------------------------------------------
# random-field helpers
# --------------------------------------------------------------------------------------

def grf(shape, ell, rng):
    """Unit-variance periodic Gaussian random field, correlation ~ exp(-r^2 / 2 ell^2).

    White N(0,1) noise multiplied in Fourier space by exp(-|k|^2 ell^2 / 4), renormalised
    to zero mean / unit standard deviation (SURVEY.md 8(d) `G_ell`).  shape is (.., Ny, Nx).
    """
    white = rng.standard_normal(shape)
    f = np.fft.rfftn(white)
    k2 = np.zeros(f.shape)
    nd = len(shape)
    for ax, n in enumerate(shape):
        if ax == nd - 1:
            k = 2.0 * np.pi * np.fft.rfftfreq(n)
        else:
            k = 2.0 * np.pi * np.fft.fftfreq(n)
        sh = [1] * nd
        sh[ax] = k.shape[0]
        k2 = k2 + (k.reshape(sh)) ** 2
    f *= np.exp(-k2 * (ell * ell) / 4.0)
    g = np.fft.irfftn(f, s=shape, axes=tuple(range(nd)))
    g -= g.mean()
    s = g.std()
    if s > 0:
        g /= s
    return g


def _brick_expand(brick_arr, b):
    """Repeat a per-brick array to per-voxel resolution."""
    out = brick_arr
    for ax in range(brick_arr.ndim):
        out = np.repeat(out, b, axis=ax)
    return out


def dirs_2d(n, phase=0.5):
    """theta_k = 2 pi (k + phase) / n ; w = 1/n."""
    th = 2.0 * np.pi * (np.arange(n) + phase) / n
    d = np.stack([np.cos(th), np.sin(th)], axis=1).astype(np.float32)
    w = np.full(n, 1.0 / n, dtype=np.float32)
    return d, w


def gauss_radau_unit(n):
    """n-point Gauss-Radau rule on mu in [0, 1] with the fixed node at mu = 0: returns (mu, w), sum w = 1, exact for
    polynomials of degree <= 2n - 2.  Interior nodes are the roots of (P_{n-1}(x) + P_n(x)) / (1 + x) on [-1, 1],
    weights (1 - x) / (n^2 P_{n-1}(x)^2) and 2 / n^2 at x = -1 (computed numerically, not tabulated)."""
    from numpy.polynomial import legendre as L
    c = np.zeros(n + 1)
    c[n - 1] = c[n] = 1.0
    roots = L.legroots(c)
    x = np.sort(np.real(roots))
    x[0] = -1.0
    pn1 = L.legval(x, np.eye(n)[n - 1])
    w = (1.0 - x) / (n * n * pn1 * pn1)
    w[0] = 2.0 / (n * n)
    return (x + 1.0) / 2.0, w / 2.0


def dirs_25d(n_phi, n_incl=4, phase=0.5):
    """2.5D quadrature of PAPER.md:347: n_phi in-plane azimuths x an n_incl-point Gauss-Radau rule in mu = cos(theta),
    theta the angle to the homogeneous out-of-plane axis (mu = 0: in-plane rays).  Returns in-plane unit directions
    [n_phi * n_incl][2], weights (sum 1; the hemisphere mu < 0 mirrors mu > 0) and sin(theta) per direction."""
    d2, _ = dirs_2d(n_phi, phase=phase)
    mu, w = gauss_radau_unit(n_incl)
    dirs = np.repeat(d2, n_incl, axis=0)
    weights = np.tile(w, n_phi) / float(n_phi)
    sin_incl = np.tile(np.sqrt(1.0 - mu * mu), n_phi)
    return (np.ascontiguousarray(dirs, dtype=np.float32), weights.astype(np.float32), sin_incl.astype(np.float32))


def dirs_fibonacci(n):
    """Spherical Fibonacci lattice z_k = 1-(2k+1)/n, phi_k = k pi (3 - sqrt 5)."""
    k = np.arange(n)
    z = 1.0 - (2.0 * k + 1.0) / n
    phi = k * np.pi * (3.0 - np.sqrt(5.0))
    r = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    d = np.stack([r * np.cos(phi), r * np.sin(phi), z], axis=1).astype(np.float32)
    w = np.full(n, 1.0 / n, dtype=np.float32)
    return d, w


def probes_every(dims, ndim, stride=1):
    """Probe at the centre of every `stride`-th voxel per axis, x fastest ordering."""
    nx, ny, nz = dims
    xs = np.arange(0, nx, stride, dtype=np.float64) + 0.5
    ys = np.arange(0, ny, stride, dtype=np.float64) + 0.5
    if ndim == 2:
        yy, xx = np.meshgrid(ys, xs, indexing="ij")
        p = np.stack([xx.ravel(), yy.ravel()], axis=1)
    else:
        zs = np.arange(0, nz, stride, dtype=np.float64) + 0.5
        zz, yy, xx = np.meshgrid(zs, ys, xs, indexing="ij")
        p = np.stack([xx.ravel(), yy.ravel(), zz.ravel()], axis=1)
    return np.ascontiguousarray(p.astype(np.float32))


def sample_probes(probe_pos, n, seed):
    """Seeded subset of probes (sorted, so neighbours stay neighbours)."""
    if n >= probe_pos.shape[0]:
        return probe_pos
    rng = np.random.default_rng(seed)
    idx = np.sort(rng.choice(probe_pos.shape[0], size=n, replace=False))
    return np.ascontiguousarray(probe_pos[idx])


def _brick_classes(rng, occ_b, probs=(0.4, 0.2, 0.2, 0.2)):
    """Seeded class 0..3 per brick; bricks touching an empty brick are forced 'rough' (3)."""
    cls = rng.choice(4, size=occ_b.shape, p=list(probs))
    emp = ~occ_b
    touch = np.zeros_like(occ_b)
    for ax in range(occ_b.ndim):
        for sh in (-1, 1):
            touch |= np.roll(emp, sh, axis=ax)
    cls[touch & occ_b] = 3
    return cls


_CLASS_AF = np.array([[0.0, 0.0], [0.3, 0.0], [0.6, 0.0], [0.0, 0.5]])


def _planck_ratio(T, lam_nm=500.0, Tref=4000.0):
    x = 1.438776877e7 / lam_nm  # hc/(lambda k) in K for lambda in nm
    return (np.exp(x / Tref) - 1.0) / (np.exp(x / T) - 1.0)


# --------------------------------------------------------------------------------------
# configs
# --------------------------------------------------------------------------------------

def _c1(n, n_dirs, rng):
    nl = 8
    chi0 = np.exp(np.log(1e-3) + 1.0 * rng.standard_normal((n, n)))
    S = np.exp(0.5 * rng.standard_normal((n, n)))
    j = np.arange(nl)
    prof = np.exp(-((j - 3.5) / 2.0) ** 2)
    chi = chi0[..., None] * prof
    eta = chi * S[..., None]
    d, w = dirs_2d(n_dirs)
    wl = Workload(
        name="C1", ndim=2, dims=(n, n, 1), brick=16, voxel_size=1.0,
        active=np.ones(n * n, dtype=np.uint8), variant=VARIANT_ISO, n_lambda=nl, lambda_batch=8,
        max_level=0, metric=METRIC_RELVAR, thr_eta=0.0, thr_chi=0.0, tau_gate=-1.0,
        probe_pos=probes_every((n, n, 1), 2), dirs=d, weights=w,
        eta=np.ascontiguousarray(eta.reshape(n * n, nl).astype(np.float32)),
        chi=np.ascontiguousarray(chi.reshape(n * n, nl).astype(np.float32)),
    )
    return wl


def _occupancy_top(gb, n_keep):
    """Occupied = the n_keep bricks with the largest field value."""
    flat = gb.ravel()
    order = np.argsort(-flat, kind="stable")
    occ = np.zeros(flat.shape, dtype=bool)
    occ[order[:n_keep]] = True
    return occ.reshape(gb.shape)


def _c2(n, n_dirs, rng, n_lambda=32, max_level=3):
    b = 16
    nb = n // b
    sc = n / 512.0
    occ_b = _occupancy_top(grf((nb, nb), 3.0 * max(sc, 0.25), rng), int(round(0.4 * nb * nb)))
    cls = _brick_classes(rng, occ_b)
    A = _brick_expand(_CLASS_AF[cls, 0], b)
    F = _brick_expand(_CLASS_AF[cls, 1], b)
    occ = _brick_expand(occ_b, b)
    ln_chi_l = (np.log(5e-2) + 1.5 * grf((n, n), 48.0 * sc, rng) + A * grf((n, n), 6.0 * sc, rng)
                + F * rng.standard_normal((n, n)))
    chi_l = np.exp(ln_chi_l)
    chi_c = 5e-4 * np.exp(0.5 * grf((n, n), 96.0 * sc, rng))
    S = np.exp(0.5 * grf((n, n), 64.0 * sc, rng))
    j = np.arange(n_lambda)
    prof = np.exp(-((j - (n_lambda - 1) / 2.0) / (n_lambda / 8.0)) ** 2)
    chi = chi_c[..., None] + chi_l[..., None] * prof
    eta = chi * S[..., None]
    chi[~occ] = 0.0
    eta[~occ] = 0.0
    d, w = dirs_2d(n_dirs)
    return Workload(
        name="C2", ndim=2, dims=(n, n, 1), brick=b, voxel_size=1.0,
        active=occ.astype(np.uint8).ravel(), variant=VARIANT_ISO, n_lambda=n_lambda, lambda_batch=8,
        max_level=max_level, metric=METRIC_RELVAR, thr_eta=1e-2, thr_chi=1e-2, tau_gate=-1.0,
        probe_pos=probes_every((n, n, 1), 2), dirs=d, weights=w,
        eta=np.ascontiguousarray(eta.reshape(n * n, n_lambda).astype(np.float32)),
        chi=np.ascontiguousarray(chi.reshape(n * n, n_lambda).astype(np.float32)),
    )


def _solar_base(n, rng):
    """Stratified solar-like 2D atmosphere shared by C3 and C4."""
    b = 16
    nb = n // b
    sc = n / 1024.0
    y = np.arange(n, dtype=np.float64)[:, None] * np.ones((1, n))
    # sparsity: upper 40 % of brick rows is 75 % empty by blobs, below all active
    row0 = int(round(0.6 * nb))  # 38 of 64 (0.59375) -> use the survey's 38/64 proportion
    if nb == 64:
        row0 = 38
    occ_b = np.ones((nb, nb), dtype=bool)
    n_up = (nb - row0) * nb
    gb = grf((nb, nb), 3.0 * max(sc, 0.25), rng)
    up = np.zeros((nb, nb), dtype=bool)
    up[row0:, :] = True
    vals = np.where(up, gb, -np.inf)
    keep = _occupancy_top(vals, int(round(0.25 * n_up)))
    occ_b[up] = keep[up]
    occ = _brick_expand(occ_b, b)
    chi_lc = 10.0 * 10.0 ** (-6.0 * y / (n - 1)) * np.exp(0.2 * grf((n, n), 16.0 * sc, rng))
    mid = (n - 1) / 2.0
    T = np.where(y < mid, 4000.0 + 2000.0 * ((mid - y) / mid) ** 2,
                 4000.0 + 6000.0 * ((y - mid) / (n - 1 - mid)) ** 2)
    S = _planck_ratio(T)
    vx = 20.0 * grf((n, n), 24.0 * sc, rng)
    vy = 20.0 * grf((n, n), 24.0 * sc, rng)
    vth = 12.85 * np.sqrt(T / 1.0e4)
    return dict(b=b, occ=occ, chi_lc=chi_lc, T=T, S=S, vx=vx, vy=vy, vth=vth)


def _line_fields(base, lam0, strength, width_fac):
    dlamD = lam0 * base["vth"] * width_fac / C_LIGHT_KMS
    chi_star = strength * base["chi_lc"] * np.sqrt(np.pi) * dlamD
    eta_star = chi_star * base["S"]
    a0 = np.full_like(chi_star, 0.01)
    return eta_star, chi_star, a0, 1.0 / dlamD


def _zero_inactive(arrs, occ):
    for a in arrs:
        a[~occ] = 0.0


def _c3(n, n_dirs, rng, n_lambda=64, max_level=4, n_vbins=8):
    base = _solar_base(n, rng)
    occ = base["occ"]
    lam0 = 500.0
    lam = (lam0 * (1.0 + np.linspace(-120.0, 120.0, n_lambda) / C_LIGHT_KMS)).astype(np.float32)
    es, cs, a0, inv = _line_fields(base, lam0, 1.0, 1.0)
    chi_bg1 = 1e-3 * base["chi_lc"]
    eta_bg1 = chi_bg1 * base["S"]
    vel = np.stack([base["vx"], base["vy"]], axis=-1)
    _zero_inactive([es, cs, a0, inv, chi_bg1, eta_bg1, vel], occ)
    nv = n * n
    chi_bg = np.repeat(chi_bg1.reshape(nv, 1), n_lambda, axis=1)
    eta_bg = np.repeat(eta_bg1.reshape(nv, 1), n_lambda, axis=1)
    d, w = dirs_2d(n_dirs)
    nbatch = n_lambda // 8
    al = np.full((nbatch, 4), -1, dtype=np.int8)
    al[:, 0] = 0
    f32 = lambda x: np.ascontiguousarray(x.astype(np.float32))
    return Workload(
        name="C3", ndim=2, dims=(n, n, 1), brick=16, voxel_size=1.0, active=occ.astype(np.uint8).ravel(),
        variant=VARIANT_VELINTERP, n_lambda=n_lambda, lambda_batch=8, max_level=max_level,
        metric=METRIC_RELVAR, thr_eta=1e-2, thr_chi=1e-2, tau_gate=-1.0,
        probe_pos=probes_every((n, n, 1), 2), dirs=d, weights=w,
        lam=lam, eta_bg=f32(eta_bg), chi_bg=f32(chi_bg), vel=f32(vel.reshape(nv, 2)),
        n_lines=1, lambda0=np.array([lam0], dtype=np.float32),
        eta_star0=f32(es.reshape(1, nv)), chi_star0=f32(cs.reshape(1, nv)),
        a0=f32(a0.reshape(1, nv)), inv_dlamD=f32(inv.reshape(1, nv)),
        active_lines=al, n_vbins=n_vbins,
    )


def _c4(n, n_dirs, rng, n_line_lambda=64, n_cont=16, max_level=4):
    base = _solar_base(n, rng)
    occ = base["occ"]
    lam0s = [500.0, 500.1, 600.0]
    strengths = [1.0, 0.3, 0.1]
    widths = [1.0, 1.0, 0.5]
    nv = n * n
    lam_parts, fields = [], []
    for l0, s, wf in zip(lam0s, strengths, widths):
        lam_parts.append(l0 * (1.0 + np.linspace(-120.0, 120.0, n_line_lambda) / C_LIGHT_KMS))
        fields.append(_line_fields(base, l0, s, wf))
    # continuum wavelengths in 420-580 nm, outside every line window
    cont = np.linspace(420.0, 580.0, n_cont + 2)[1:-1]
    for l0 in lam0s:
        lo, hi = l0 * (1 - 120.0 / C_LIGHT_KMS), l0 * (1 + 120.0 / C_LIGHT_KMS)
        cont = np.where((cont >= lo - 0.5) & (cont <= hi + 0.5), cont + 1.7, cont)
    lam_parts.append(cont)
    lam = np.concatenate(lam_parts).astype(np.float32)
    n_lambda = lam.shape[0]
    assert n_lambda % 8 == 0
    chi_bg = 1e-3 * base["chi_lc"].reshape(nv, 1) * (lam.astype(np.float64)[None, :] / 500.0) ** 3
    eta_bg = chi_bg * base["S"].reshape(nv, 1)
    vel = np.stack([base["vx"], base["vy"]], axis=-1).reshape(nv, 2)
    occv = occ.ravel()
    chi_bg[~occv] = 0.0
    eta_bg[~occv] = 0.0
    vel[~occv] = 0.0
    es = np.stack([f[0].ravel() for f in fields])
    cs = np.stack([f[1].ravel() for f in fields])
    a0 = np.stack([f[2].ravel() for f in fields])
    inv = np.stack([f[3].ravel() for f in fields])
    for a in (es, cs, a0, inv):
        a[:, ~occv] = 0.0
    nbatch = n_lambda // 8
    al = np.full((nbatch, 4), -1, dtype=np.int8)
    per = n_line_lambda // 8
    for bi in range(nbatch):
        if bi < 2 * per:
            al[bi, 0], al[bi, 1] = 0, 1      # blended pair 500.0 / 500.1 nm
        elif bi < 3 * per:
            al[bi, 0] = 2
    d, w = dirs_2d(n_dirs)
    f32 = lambda x: np.ascontiguousarray(x.astype(np.float32))
    return Workload(
        name="C4", ndim=2, dims=(n, n, 1), brick=16, voxel_size=1.0, active=occ.astype(np.uint8).ravel(),
        variant=VARIANT_CAV, n_lambda=n_lambda, lambda_batch=8, max_level=max_level,
        metric=METRIC_RELVAR, thr_eta=1e-2, thr_chi=1e-2, tau_gate=-1.0,
        probe_pos=probes_every((n, n, 1), 2), dirs=d, weights=w,
        lam=lam, eta_bg=f32(eta_bg), chi_bg=f32(chi_bg), vel=f32(vel),
        n_lines=3, lambda0=np.array(lam0s, dtype=np.float32),
        eta_star0=f32(es), chi_star0=f32(cs), a0=f32(a0), inv_dlamD=f32(inv),
        active_lines=al, n_vbins=0,
    )


# C5 brick classes (smooth / mild / structured / rough): small-scale amplitudes (A of G_4, F of white noise) in ln chi and
# the small-scale share of the velocity field.  Round 2 retune (SURVEY.md 8(d) allows it, "stating so"): with the round-1
# recipe (ln chi on 24 voxels, velocities on 16, scale height 12) the eq. 17 Core-and-Voigt test left 99.4 % of the
# populated bricks at level 0, so the config timed brick skipping only; a 20 km/s field must vary on >~ 100 voxels for
# 2^3 / 4^3 cells to pass at relative variance 1e-2 (the Gaussian core turns dv into d ln(phi) = 2 x dv / v_th).
_C5_CLASS_AF = np.array([[0.0, 0.0], [0.1, 0.0], [0.4, 0.0], [0.0, 0.5]])
_C5_CLASS_VEL = (0.0, 0.005, 0.05, 0.2)
_C5_CLASS_P = (0.5, 0.3, 0.1, 0.1)


def _c5(n, n_dirs, rng, n_lambda=32, max_level=2, probe_stride=4, lnf_len=128.0, vel_len=128.0, hs0=48.0, s_len=96.0,
        vel_small=_C5_CLASS_VEL, cls_af=_C5_CLASS_AF, cls_p=_C5_CLASS_P):
    b = 8
    nb = n // b
    sc = n / 256.0
    # warped-slab occupancy on the brick lattice: smallest |z_b - nb/2 + (nb/8) G_4(x_b,y_b)|
    g4 = grf((nb, nb), 4.0 * max(sc, 0.25), rng)
    zb = np.arange(nb, dtype=np.float64)[:, None, None]
    dist = np.abs(zb - nb / 2.0 + (nb / 8.0) * g4[None, :, :])
    occ_b = _occupancy_top(-dist, int(round(0.3 * nb ** 3)))
    cls = _brick_classes(rng, occ_b, cls_p)
    caf = np.asarray(cls_af, dtype=np.float64)
    A = _brick_expand(caf[cls, 0], b)
    F = _brick_expand(caf[cls, 1], b)
    occ = _brick_expand(occ_b, b)
    zs = n / 2.0 + (n / 8.0) * grf((n, n), 32.0 * sc, rng)          # z_s(x, y)
    z = np.arange(n, dtype=np.float64)[:, None, None]
    dz = np.abs(z - zs[None, :, :])
    sh = (n, n, n)
    lnf = 1.5 * grf(sh, lnf_len * sc, rng) + A * grf(sh, 4.0 * sc, rng) + F * rng.standard_normal(sh)
    hs = hs0 * sc
    chi_lc = 0.3 * np.exp(-dz / hs) * np.exp(lnf)
    del lnf
    S = (1.0 + 2.0 * np.exp(-dz / hs)) * np.exp(0.3 * grf(sh, s_len * sc, rng))
    Av = _brick_expand(np.asarray(vel_small, dtype=np.float64)[cls], b)
    vel = np.stack([20.0 * (np.sqrt(1.0 - Av * Av) * grf(sh, vel_len * sc, rng) + Av * grf(sh, 4.0 * sc, rng))
                    for _ in range(3)], axis=-1)
    T = 6000.0 + 2000.0 * np.exp(-dz / hs)
    vth = 12.85 * np.sqrt(T / 1.0e4)
    lam0 = 500.0
    lam = (lam0 * (1.0 + np.linspace(-90.0, 90.0, n_lambda) / C_LIGHT_KMS)).astype(np.float32)
    dlamD = lam0 * vth / C_LIGHT_KMS
    cs = chi_lc * np.sqrt(np.pi) * dlamD
    es = cs * S
    a0 = np.full(sh, 0.01)
    inv = 1.0 / dlamD
    chi_bg1 = 1e-3 * chi_lc
    eta_bg1 = chi_bg1 * S
    _zero_inactive([es, cs, a0, inv, chi_bg1, eta_bg1, vel], occ)
    nv = n ** 3
    f32 = lambda x: np.ascontiguousarray(x.astype(np.float32))
    chi_bg = np.repeat(f32(chi_bg1.reshape(nv, 1)), n_lambda, axis=1)
    eta_bg = np.repeat(f32(eta_bg1.reshape(nv, 1)), n_lambda, axis=1)
    d, w = dirs_fibonacci(n_dirs)
    nbatch = n_lambda // 8
    al = np.full((nbatch, 4), -1, dtype=np.int8)
    al[:, 0] = 0
    return Workload(
        name="C5", ndim=3, dims=(n, n, n), brick=b, voxel_size=1.0, active=occ.astype(np.uint8).ravel(),
        variant=VARIANT_CAV, n_lambda=n_lambda, lambda_batch=8, max_level=max_level,
        metric=METRIC_RELVAR, thr_eta=1e-2, thr_chi=1e-2, tau_gate=-1.0,
        probe_pos=probes_every((n, n, n), 3, stride=probe_stride), dirs=d, weights=w,
        lam=lam, eta_bg=np.ascontiguousarray(eta_bg), chi_bg=np.ascontiguousarray(chi_bg),
        vel=f32(vel.reshape(nv, 3)),
        n_lines=1, lambda0=np.array([lam0], dtype=np.float32),
        eta_star0=f32(es.reshape(1, nv)), chi_star0=f32(cs.reshape(1, nv)),
        a0=f32(a0.reshape(1, nv)), inv_dlamD=f32(inv.reshape(1, nv)),
        active_lines=al, n_vbins=0, notes={"brick_class": cls},
    )


_FULL = {
    "C1": dict(n=64, n_dirs=16),
    "C2": dict(n=512, n_dirs=64),
    "C3": dict(n=1024, n_dirs=64),
    "C4": dict(n=1024, n_dirs=128),
    "C5": dict(n=256, n_dirs=48),
}


def make(name: str, n: Optional[int] = None, n_dirs: Optional[int] = None,
         n_probes: Optional[int] = None, seed: Optional[int] = None, **kw) -> Workload:
    """Build config `name` ('C1'..'C5').  `n` / `n_dirs` shrink the grid / quadrature for tests
    (field length scales shrink with n); `n_probes` keeps a seeded, sorted probe subset."""
    if name not in _FULL:
        raise ValueError(f"unknown config {name}")
    full = _FULL[name]
    n = full["n"] if n is None else int(n)
    n_dirs = full["n_dirs"] if n_dirs is None else int(n_dirs)
    seed = SEEDS[name] if seed is None else int(seed)
    rng = np.random.default_rng(seed)
    fn = {"C1": _c1, "C2": _c2, "C3": _c3, "C4": _c4, "C5": _c5}[name]
    wl = fn(n, n_dirs, rng, **kw)
    wl.notes["seed"] = seed
    wl.notes["n_probes_full"] = int(wl.probe_pos.shape[0])
    if n_probes is not None:
        wl.probe_pos = sample_probes(wl.probe_pos, int(n_probes), seed + 17)
    return wl


def batch_workload(wl, batches):
    """The same atmosphere and rays restricted to the wavelength batches `batches` (a list of batch indices): pure
    column selection, returns (workload, wavelength indices).  Batches are independent (one level table per batch,
    PAPER.md:351; pinned by test_batches_are_independent_in_the_oracle), so the oracle's pyramid, level table, lists, I
    and J of the restricted workload are those columns / rows of the full one: this is how the BASELINE-size configs
    are compared with (and bench.py's cpu_baseline is timed on) the oracle without a numpy build of every batch."""
    import copy
    W = wl.lambda_batch
    idx = np.concatenate([np.arange(b * W, (b + 1) * W) for b in batches])
    out = copy.copy(wl)
    out.n_lambda = int(idx.size)
    for name in ("eta", "chi", "eta_bg", "chi_bg"):
        a = getattr(wl, name)
        if a is not None:
            setattr(out, name, np.ascontiguousarray(a[:, idx]))
    if wl.lam is not None:
        out.lam = np.ascontiguousarray(wl.lam[idx])
    if wl.active_lines is not None:
        out.active_lines = np.ascontiguousarray(wl.active_lines[list(batches)])
    if wl.i0 is not None:
        out.i0 = np.ascontiguousarray(wl.i0[:, idx])
    return out, idx
