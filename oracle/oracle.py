"""Python face of the CPU ORACLE (test infrastructure -- never imported by the product).

Marches and the Voigt function are the plain C in dex_oracle.c (fp64).  The mip pyramid,
the VLM cell test and the per-brick level selection are written out here in numpy, in fp64,
following SURVEY.md 8(c) V-rules (restated in DESIGN.md) and the passages cited per function.
Nothing here imports, links or reads anything of paper_2511_08498_b200/.
"""
from __future__ import annotations

import ctypes as C
import math
from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

from . import build as _build

_LIB = None
MAX_LINES = 4

ISO, VELINTERP, CAV, CLASSIC = 0, 1, 2, 3
IOD_LOG, RELVAR = 0, 1


class _Grid(C.Structure):
    _fields_ = [("ndim", C.c_int), ("dims", C.c_int * 3), ("brick", C.c_int), ("h", C.c_double),
                ("n_caps", C.c_int), ("cap_t", C.c_float * 8), ("sin_incl", C.c_void_p),
                ("t_begin", C.c_float), ("t_end", C.c_float)]


_PP = C.POINTER(C.c_void_p)


class _Fields(C.Structure):
    _fields_ = [
        ("variant", C.c_int), ("n_lambda", C.c_int), ("W", C.c_int), ("n_levels", C.c_int),
        ("eta", _PP), ("chi", _PP), ("lam", C.c_void_p), ("n_lines", C.c_int), ("lambda0", C.c_void_p),
        ("eta_star", _PP), ("chi_star", _PP), ("a0", _PP), ("inv_dlamD", _PP), ("vbar", _PP),
        ("active_lines", C.c_void_p), ("c_light", C.c_double), ("n_vbins", C.c_int),
        ("vtab", _PP), ("vmax", _PP),
    ]


class _Capture(C.Structure):
    _fields_ = [("counts", C.c_void_p), ("records", C.c_void_p), ("ds", C.c_void_p),
                ("cap_stride", C.c_int), ("batch", C.c_int)]


def lib():
    global _LIB
    if _LIB is None:
        L = C.CDLL(_build.build())
        L.orc_segment.restype = C.c_double
        L.orc_segment.argtypes = [C.c_double] * 4
        L.orc_voigt_H.restype = C.c_double
        L.orc_voigt_H.argtypes = [C.c_double] * 2
        L.orc_voigt_H_array.restype = None
        L.orc_voigt_H_array.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64]
        L.orc_line_terms.restype = None
        L.orc_line_terms.argtypes = [C.c_double] * 8 + [C.POINTER(C.c_double)] * 2
        L.orc_plain_march.restype = C.c_int64
        L.orc_plain_march.argtypes = [C.POINTER(_Grid), C.POINTER(_Fields), C.c_int64, C.c_void_p, C.c_int,
                                      C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(_Capture), C.c_int]
        L.orc_hdda_march.restype = C.c_int64
        L.orc_hdda_march.argtypes = [C.POINTER(_Grid), C.POINTER(_Fields), C.c_void_p, C.c_int64, C.c_void_p,
                                     C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(_Capture), C.c_int]
        L.orc_mean_intensity.restype = None
        L.orc_mean_intensity.argtypes = [C.c_int64, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_max_threads.restype = C.c_int
        L.orc_init.restype = None
        L.orc_init()
        _LIB = L
    return _LIB


def max_threads() -> int:
    return int(lib().orc_max_threads())


# --------------------------------------------------------------------------------------
# scalar pieces
# --------------------------------------------------------------------------------------

def segment(I_in, eta, chi, hds):
    """eq. 3 with constant eta, chi over a path h*ds."""
    return lib().orc_segment(float(I_in), float(eta), float(chi), float(hds))


def voigt_H(a, x):
    """H(a,x) by HUM1WEI24; scalars or arrays."""
    a = np.asarray(a, dtype=np.float64)
    x = np.asarray(x, dtype=np.float64)
    a, x = np.broadcast_arrays(a, x)
    a = np.ascontiguousarray(a)
    x = np.ascontiguousarray(x)
    out = np.empty(a.shape, dtype=np.float64)
    lib().orc_voigt_H_array(a.ctypes.data, x.ctypes.data, out.ctypes.data, a.size)
    return out


def line_terms(lam, lam0, eta_star0, chi_star0, a0, inv_dlamD, vproj, c_light):
    """eqs. 14-20 for arrays (numpy broadcast); returns (eta_l, chi_l) in fp64.  Same arithmetic,
    in the same order, as orc_line_terms in dex_oracle.c (which the marches call)."""
    lam = np.asarray(lam, dtype=np.float64)
    x = ((lam - lam0) + (np.asarray(vproj, dtype=np.float64) / c_light) * lam0) * np.asarray(inv_dlamD, np.float64)
    r = lam / lam0
    a = r * r * np.asarray(a0, np.float64)
    a, x = np.broadcast_arrays(a, x)
    phi = voigt_H(a, x) * np.asarray(inv_dlamD, np.float64) / math.sqrt(math.pi)
    s = lam0 / lam
    return s * np.asarray(eta_star0, np.float64) * phi, s * np.asarray(chi_star0, np.float64) * phi


# --------------------------------------------------------------------------------------
# grid helpers
# --------------------------------------------------------------------------------------

def grid_shape(wl, m=0):
    """numpy shape (.., Ny_m, Nx_m) of the level-m grid."""
    nx, ny, nz = wl.dims
    if wl.ndim == 2:
        return (ny >> m, nx >> m)
    return (nz >> m, ny >> m, nx >> m)


def brick_active(wl) -> np.ndarray:
    """Brick is populated iff any of its voxels is active. bool [n_bricks]."""
    b = wl.brick
    act = wl.active.reshape(grid_shape(wl)).astype(bool)
    if wl.ndim == 2:
        ny, nx = act.shape
        return act.reshape(ny // b, b, nx // b, b).any(axis=(1, 3)).ravel()
    nz, ny, nx = act.shape
    return act.reshape(nz // b, b, ny // b, b, nx // b, b).any(axis=(1, 3, 5)).ravel()


def children(arr, ndim):
    """The 2^D children of every parent cell as strided views, in child order: x fastest, then y,
    then z.  arr has shape (.., Ny, Nx, channels...)."""
    out = []
    if ndim == 2:
        for dy in (0, 1):
            for dx in (0, 1):
                out.append(arr[dy::2, dx::2])
    else:
        for dz in (0, 1):
            for dy in (0, 1):
                for dx in (0, 1):
                    out.append(arr[dz::2, dy::2, dx::2])
    return out


def mip_mean(arr, ndim):
    """V1: box filter: parent = mean of its 2^D children, summed in fp64 in child
    order, multiplied by 2^-D (exact), rounded once to fp32."""
    ch = children(arr, ndim)
    acc = ch[0].astype(np.float64)
    for c in ch[1:]:
        acc = acc + c.astype(np.float64)
    acc = acc * (1.0 / len(ch))
    return acc.astype(np.float32)


def mip_max(arr, ndim):
    ch = children(arr, ndim)
    acc = ch[0]
    for c in ch[1:]:
        acc = np.maximum(acc, c)
    return acc


def cell_metric(ch64: List[np.ndarray], metric: int, h: float):
    """V2/V4: statistic of one quantity over the 2^D children of every parent cell (fp64).
    RELVAR : Var[x]/Mean[x]^2 of the raw values.
    IOD_LOG: |Var[X]/Mean[X]|, X = ln(x h)  (eq. 8), population variance.
    Children all exactly equal -> 0.  IOD_LOG with any child <= 0 and not all equal -> +inf."""
    n = len(ch64)
    all_equal = np.ones(ch64[0].shape, dtype=bool)
    for c in ch64[1:]:
        all_equal &= (c == ch64[0])
    with np.errstate(all="ignore"):
        if metric == IOD_LOG:
            bad = np.zeros(ch64[0].shape, dtype=bool)
            for c in ch64:
                bad |= ~(c > 0.0)
            X = [np.log(c * h) for c in ch64]
        else:
            bad = None
            X = ch64
        s = X[0].copy()
        for c in X[1:]:
            s = s + c
        mean = s / n
        d = X[0] - mean
        v = d * d
        for c in X[1:]:
            d = c - mean
            v = v + d * d
        var = v / n
        if metric == IOD_LOG:
            val = np.abs(var / mean)
        else:
            val = var / (mean * mean)
    val = np.where(np.isnan(val), np.inf, val)
    if bad is not None:
        val = np.where(bad, np.inf, val)
    val = np.where(all_equal, 0.0, val)
    return val


def raw_mean(ch64):
    s = ch64[0].copy()
    for c in ch64[1:]:
        s = s + c
    return s / len(ch64)


def pack_levels(levels_row: np.ndarray, max_level: int) -> np.ndarray:
    """state = level+1 (0 = empty) in ceil(log2(max_level+2)) bits, floor(64/bits)
    bricks per 64-bit word, no straddling."""
    bits = max(1, math.ceil(math.log2(max_level + 2)))
    per = 64 // bits
    n = levels_row.shape[0]
    words = np.zeros((n + per - 1) // per, dtype=np.uint64)
    for i in range(n):
        words[i // per] |= np.uint64(int(levels_row[i]) + 1) << np.uint64((i % per) * bits)
    return words


# --------------------------------------------------------------------------------------
# mips + VLM level selection
# --------------------------------------------------------------------------------------

@dataclass
class OracleMips:
    wl: object
    variant: int
    max_level: int
    levels: np.ndarray                      # int8 [n_batch][n_bricks]
    eta: List[np.ndarray] = field(default_factory=list)   # per level [cells][n_lambda] (ISO eta / bg)
    chi: List[np.ndarray] = field(default_factory=list)
    eta_star: List[np.ndarray] = field(default_factory=list)  # per level [n_lines][cells]
    chi_star: List[np.ndarray] = field(default_factory=list)
    a0: List[np.ndarray] = field(default_factory=list)
    inv_dlamD: List[np.ndarray] = field(default_factory=list)
    vbar: List[np.ndarray] = field(default_factory=list)      # per level [cells][ndim]
    vmax: List[np.ndarray] = field(default_factory=list)      # per level [cells]
    vtab: List[np.ndarray] = field(default_factory=list)      # per level [cells][n_vbins][n_lambda][2]
    cell_pass: List[np.ndarray] = field(default_factory=list)  # per level m>=1: bool [cells_m][n_batch]


def _to_grid(wl, flat, m, trailing):
    return flat.reshape(grid_shape(wl, m) + tuple(trailing))


def _velinterp_at(tab, V, v, n_vbins):
    """Interpolate tables tab[..., n_vbins, n_lambda, 2] (fp32) at velocity v (array over cells) on the
    uniform grid [-V, V], clamped (same rule as velinterp_lookup in dex_oracle.c)."""
    V = V.astype(np.float64)
    with np.errstate(all="ignore"):
        f = (v + V) / (2.0 * V) * float(n_vbins - 1)
    f = np.where(V > 0.0, f, 0.0)
    f = np.clip(f, 0.0, float(n_vbins - 1))
    i0 = np.minimum(np.floor(f).astype(np.int64), n_vbins - 2)
    w = f - i0
    idx0 = i0[..., None, None, None]
    t0 = np.take_along_axis(tab, idx0, axis=-3)[..., 0, :, :].astype(np.float64)
    t1 = np.take_along_axis(tab, idx0 + 1, axis=-3)[..., 0, :, :].astype(np.float64)
    ww = w[..., None, None]
    return (1.0 - ww) * t0 + ww * t1


def _line_sum(wl, lam_idx, lines, es, cs, a0, inv, vproj_per_line, bg_eta, bg_chi):
    """eqs. 10-11: background + sum over the active lines, for wavelength indices lam_idx.
    es/cs/a0/inv: [n_lines][cells...]; vproj_per_line: dict line -> array[cells..., len(lam_idx)] or
    array[cells...]; returns fp64 arrays [cells..., len(lam_idx)]."""
    lam = wl.lam[lam_idx].astype(np.float64)
    e = bg_eta.astype(np.float64).copy()
    c = bg_chi.astype(np.float64).copy()
    for l in lines:
        vp = vproj_per_line[l]
        if vp.ndim == es[l].ndim:
            vp = vp[..., None]
        el, cl = line_terms(lam, float(wl.lambda0[l]), es[l][..., None], cs[l][..., None], a0[l][..., None],
                            inv[l][..., None], vp, wl.c_light)
        e = e + el
        c = c + cl
    return e, c


def velinterp_parent_table(child_tabs, child_V, Vp, n_vbins):
    """DESIGN.md reading R-vel (the construction of the higher levels is not stated): the parent's
    velocity grid is uniform on [-Vp, Vp], Vp = max over its children; its bin value is the mean, over the 2^D
    children in child order, of the CHILD's table linearly interpolated on the CHILD's own grid [-V_child, V_child]
    at the parent's bin velocity (clamped to the child's range).  child_tabs: 2^D arrays [cells..., n_vbins,
    n_lambda, 2] fp32; child_V: 2^D arrays [cells...]; Vp: [cells...].  Returns fp32 [cells..., n_vbins, n_lambda, 2]."""
    n = n_vbins
    Vp = Vp.astype(np.float64)
    tab = np.zeros(Vp.shape + (n,) + child_tabs[0].shape[-2:], dtype=np.float32)
    for k in range(n):
        vk = -Vp + 2.0 * Vp * (float(k) / float(n - 1))
        acc = None
        for cti, cV in zip(child_tabs, child_V):
            val = _velinterp_at(cti, cV, vk, n)
            acc = val if acc is None else acc + val
        acc = acc * (1.0 / len(child_tabs))
        tab[..., k, :, :] = acc.astype(np.float32)
    return tab


def velinterp_rest_frame(tab, V, n_vbins):
    """the VLM test of the velocity-interpolation scheme sees "the values for the emissivity and opacity
    in the rest frame of each voxel (i.e. the centre of the velocity grid, with a velocity of 0)": the cell's table
    interpolated at v = 0.  Returns (eta, chi) fp64 [cells..., n_lambda]."""
    z = np.zeros(V.shape, dtype=np.float64)
    t = _velinterp_at(tab, V, z, n_vbins)
    return t[..., 0], t[..., 1]


def cav_worst_case_shift(lam, lam0, V, c_light):
    """eq. 17: the Doppler shift v_D in [-V, V] that minimises |lam0 (1 - v/c) - lam|, i.e. that
    brings the line core as close to wavelength lam as the cell's velocities allow: v_D = clamp(c (1 - lam/lam0), -V, V).
    lam: [W] fp64, V: [cells...] fp64 (max |v| over the cell's voxels).  Returns [cells..., W] fp64."""
    want = c_light * (1.0 - lam / float(lam0))
    return np.clip(want, -V[..., None], V[..., None])


def cav_test_fields(wl, M, m):
    """V6: what the VLM test of the Core-and-Voigt scheme sees in the cells of level m: background
    plus the sum over the batch's active lines of the line terms (eqs. 10-20) at each cell's worst-case Doppler shift
    (eq. 17) -- "summing the emissivity and opacity from each line at a Doppler shift of v_D".  Returns (eta, chi) fp64
    [cells_m..., n_lambda]."""
    W, nl = wl.lambda_batch, wl.n_lambda
    te = np.zeros(grid_shape(wl, m) + (nl,), dtype=np.float64)
    tc = np.zeros_like(te)
    Vc = M.vmax[m].astype(np.float64)
    for b in range(wl.n_batch):
        lines = [int(l) for l in wl.active_lines[b] if l >= 0]
        idx = np.arange(b * W, (b + 1) * W)
        lam = wl.lam[idx].astype(np.float64)
        vd = {}
        for l in lines:   # eq. 17: Doppler shift closest to the line core reachable in the cell
            vd[l] = cav_worst_case_shift(lam, wl.lambda0[l], Vc, wl.c_light)     # [cells..., W]
        ee, cc = _line_sum(wl, idx, lines, M.eta_star[m], M.chi_star[m], M.a0[m], M.inv_dlamD[m], vd,
                           M.eta[m][..., idx], M.chi[m][..., idx])
        te[..., idx] = ee
        tc[..., idx] = cc
    return te, tc


def build_mips(wl, max_level=None, metric=None, thr_eta=None, thr_chi=None, tau_gate=None,
               variant=None) -> OracleMips:
    """Mip chains (V1), per-cell VLM test (V2-V4, V6) and per-brick level per batch (V5, V7).
    PAPER.md:109, :127-144, :148, :162, :188-200, :282-325, :351."""
    variant = wl.variant if variant is None else variant
    max_level = wl.max_level if max_level is None else max_level
    metric = wl.metric if metric is None else metric
    thr_eta = wl.thr_eta if thr_eta is None else thr_eta
    thr_chi = wl.thr_chi if thr_chi is None else thr_chi
    tau_gate = wl.tau_gate if tau_gate is None else tau_gate
    if variant == CLASSIC:
        max_level = 0          # brute force in every full-resolution cell
    # thresholds, gate and voxel size cross the C ABI as fp32 (include/dex.h); take them as such
    thr_eta, thr_chi, tau_gate = (float(np.float32(v)) for v in (thr_eta, thr_chi, tau_gate))
    nd, W, nl, nb = wl.ndim, wl.lambda_batch, wl.n_lambda, wl.n_batch
    h = float(np.float32(wl.voxel_size))
    B = wl.brick
    assert (1 << max_level) <= B
    act_b = brick_active(wl)
    M = OracleMips(wl=wl, variant=variant, max_level=max_level, levels=None)

    # ---- chains (V1) ----
    if variant == ISO:
        e = _to_grid(wl, wl.eta, 0, (nl,))
        c = _to_grid(wl, wl.chi, 0, (nl,))
    else:
        e = _to_grid(wl, wl.eta_bg, 0, (nl,))
        c = _to_grid(wl, wl.chi_bg, 0, (nl,))
    M.eta.append(e)
    M.chi.append(c)
    for m in range(1, max_level + 1):
        M.eta.append(mip_mean(M.eta[-1], nd))
        M.chi.append(mip_mean(M.chi[-1], nd))
    if variant != ISO:
        nL = wl.n_lines
        g0 = grid_shape(wl, 0)
        M.eta_star.append(wl.eta_star0.reshape((nL,) + g0))
        M.chi_star.append(wl.chi_star0.reshape((nL,) + g0))
        M.a0.append(wl.a0.reshape((nL,) + g0))
        M.inv_dlamD.append(wl.inv_dlamD.reshape((nL,) + g0))
        v0 = _to_grid(wl, wl.vel, 0, (nd,))
        M.vbar.append(v0)
        speed = np.sqrt((v0.astype(np.float64) ** 2).sum(axis=-1)).astype(np.float32)
        M.vmax.append(speed)
        for m in range(1, max_level + 1):
            for lst in (M.eta_star, M.chi_star, M.a0, M.inv_dlamD):
                prev = lst[-1]
                lst.append(np.stack([mip_mean(prev[l], nd) for l in range(nL)]))
            M.vbar.append(mip_mean(M.vbar[-1], nd))
            M.vmax.append(mip_max(M.vmax[-1], nd))
    if variant == VELINTERP:
        # level 0: Classic formula on the per-voxel uniform velocity grid [-|v|, |v|]
        n = wl.n_vbins
        g0 = grid_shape(wl, 0)
        tab0 = np.zeros(g0 + (n, nl, 2), dtype=np.float32)
        V0 = M.vmax[0].astype(np.float64)
        for k in range(n):
            vk = -V0 + 2.0 * V0 * (float(k) / float(n - 1))
            for b in range(nb):
                lines = [int(l) for l in wl.active_lines[b] if l >= 0]
                idx = np.arange(b * W, (b + 1) * W)
                ee, cc = _line_sum(wl, idx, lines, M.eta_star[0], M.chi_star[0], M.a0[0], M.inv_dlamD[0],
                                   {l: vk for l in lines}, M.eta[0][..., idx], M.chi[0][..., idx])
                tab0[..., k, idx, 0] = ee.astype(np.float32)
                tab0[..., k, idx, 1] = cc.astype(np.float32)
        M.vtab.append(tab0)
        for m in range(1, max_level + 1):
            # DESIGN.md reading R-vel: parent bin = mean over children of the child's table interpolated
            # at the parent's bin velocity (clamped to the child's grid)
            tab = velinterp_parent_table(children(M.vtab[-1], nd), children(M.vmax[m - 1], nd), M.vmax[m], n)
            M.vtab.append(tab)

    # ---- per-cell test (V2-V6) and brick levels (V5) ----
    n_bricks = act_b.shape[0]
    levels = np.where(act_b, 0, -1).astype(np.int8)[None, :].repeat(nb, axis=0)
    ok_so_far = np.broadcast_to(act_b, (nb, n_bricks)).copy()
    for m in range(1, max_level + 1):
        # test quantities of the children at level m-1, fp64, [cells_{m-1}][n_lambda]
        if variant == ISO:
            te, tc = M.eta[m - 1].astype(np.float64), M.chi[m - 1].astype(np.float64)
        elif variant == VELINTERP:
            te, tc = velinterp_rest_frame(M.vtab[m - 1], M.vmax[m - 1], wl.n_vbins)
        else:
            te, tc = cav_test_fields(wl, M, m - 1)
        ch_e = children(te, nd)
        ch_c = children(tc, nd)
        me = cell_metric(ch_e, metric, h)
        mc = cell_metric(ch_c, metric, h)
        ok = (me < thr_eta) & (mc < thr_chi)          # strict "<" ("IoD < 1")
        if tau_gate >= 0.0:                             # always average where chi ds is small
            ok |= (raw_mean(ch_c) * h <= tau_gate)
        # all wavelengths of a batch (V5)
        okb = ok.reshape(ok.shape[:-1] + (nb, W)).all(axis=-1)          # [cells_m][n_batch]
        M.cell_pass.append(okb)
        # all level-m cells of a brick
        cb = B >> m
        if nd == 2:
            ny, nx = okb.shape[:2]
            brick_ok = okb.reshape(ny // cb, cb, nx // cb, cb, nb).all(axis=(1, 3)).reshape(-1, nb)
        else:
            nz, ny, nx = okb.shape[:3]
            brick_ok = okb.reshape(nz // cb, cb, ny // cb, cb, nx // cb, cb, nb).all(axis=(1, 3, 5)).reshape(-1, nb)
        ok_so_far &= brick_ok.T
        levels[ok_so_far] = m
    M.levels = np.ascontiguousarray(levels)
    return M


# --------------------------------------------------------------------------------------
# marches
# --------------------------------------------------------------------------------------

def _ptr_array(arrs, keep):
    arrs = [np.ascontiguousarray(a) for a in arrs]
    keep.extend(arrs)
    pa = (C.c_void_p * max(1, len(arrs)))(*[a.ctypes.data for a in arrs])
    keep.append(pa)
    return C.cast(pa, _PP)


def _make_structs(wl, M: OracleMips, keep, level0_only=False):
    g = _Grid()
    g.ndim = wl.ndim
    for a in range(3):
        g.dims[a] = int(wl.dims[a])
    g.brick = wl.brick
    g.h = float(wl.voxel_size)
    F = _Fields()
    F.variant = M.variant
    F.n_lambda = wl.n_lambda
    F.W = wl.lambda_batch
    nlev = 1 if level0_only else (M.max_level + 1)
    F.n_levels = nlev
    F.eta = _ptr_array(M.eta[:nlev], keep)
    F.chi = _ptr_array(M.chi[:nlev], keep)
    if M.variant != ISO:
        lam = np.ascontiguousarray(wl.lam, dtype=np.float32)
        l0 = np.ascontiguousarray(wl.lambda0, dtype=np.float32)
        al = np.ascontiguousarray(wl.active_lines, dtype=np.int8)
        keep.extend([lam, l0, al])
        F.lam = lam.ctypes.data
        F.n_lines = wl.n_lines
        F.lambda0 = l0.ctypes.data
        F.active_lines = al.ctypes.data
        F.c_light = float(wl.c_light)
        F.eta_star = _ptr_array(M.eta_star[:nlev], keep)
        F.chi_star = _ptr_array(M.chi_star[:nlev], keep)
        F.a0 = _ptr_array(M.a0[:nlev], keep)
        F.inv_dlamD = _ptr_array(M.inv_dlamD[:nlev], keep)
        F.vbar = _ptr_array(M.vbar[:nlev], keep)
        F.vmax = _ptr_array(M.vmax[:nlev], keep)
        F.n_vbins = wl.n_vbins
        if M.variant == VELINTERP:
            F.vtab = _ptr_array(M.vtab[:nlev], keep)
    return g, F


@dataclass
class MarchResult:
    I: np.ndarray                 # float64 [n_probes][n_dirs][n_lambda]
    segments: int
    counts: Optional[np.ndarray] = None
    records: Optional[np.ndarray] = None
    ds: Optional[np.ndarray] = None


def _capture(n_rays, cap_stride, batch, keep):
    cap = _Capture()
    counts = np.zeros(n_rays, dtype=np.int64)
    records = np.zeros((n_rays, cap_stride), dtype=np.uint64)
    ds = np.zeros((n_rays, cap_stride), dtype=np.float32)
    keep.extend([counts, records, ds])
    cap.counts, cap.records, cap.ds = counts.ctypes.data, records.ctypes.data, ds.ctypes.data
    cap.cap_stride, cap.batch = cap_stride, batch
    return cap, counts, records, ds


def _rays(wl, probe_pos, dirs, i0):
    pp = np.ascontiguousarray(wl.probe_pos if probe_pos is None else probe_pos, dtype=np.float32)
    dd = np.ascontiguousarray(wl.dirs if dirs is None else dirs, dtype=np.float32)
    i0 = wl.i0 if i0 is None else i0
    ii = None if i0 is None else np.ascontiguousarray(i0, dtype=np.float32)
    return pp, dd, ii


def _set_interval(g, interval):
    """Finite radiance interval [t1, t2] in index units from the probe (T10); None = to the boundary."""
    if interval is None:
        return
    t1, t2 = (float(np.float32(v)) for v in interval)
    assert 0.0 <= t1 < t2
    g.t_begin, g.t_end = t1, t2


def _set_sin_incl(g, wl, dd, sin_incl, keep):
    """2.5D rays: per-direction sine of the inclination to the homogeneous axis."""
    si = getattr(wl, "sin_incl", None) if sin_incl is None else sin_incl
    if si is None:
        return
    si = np.ascontiguousarray(si, dtype=np.float32)
    assert wl.ndim == 2 and si.shape == (dd.shape[0],) and (si > 0).all() and (si <= 1).all()
    keep.append(si)
    g.sin_incl = si.ctypes.data


def plain_march(wl, M: Optional[OracleMips] = None, probe_pos=None, dirs=None, i0=None, capture=False,
                variant=None, n_threads=0, sin_incl=None, interval=None) -> MarchResult:
    """(A) AW87 DDA through every level-0 voxel; provider = fetch (ISO) or Classic."""
    if M is None:
        v = wl.variant if variant is None else variant
        v = ISO if v == ISO else CLASSIC
        M = build_mips(wl, max_level=0, variant=v)
    else:
        assert M.variant in (ISO, CLASSIC, CAV)
    keep = []
    g, F = _make_structs(wl, M, keep, level0_only=True)
    if F.variant == CAV:
        F.variant = CLASSIC
    pp, dd, ii = _rays(wl, probe_pos, dirs, i0)
    _set_sin_incl(g, wl, dd, sin_incl, keep)
    _set_interval(g, getattr(wl, "interval", None) if interval is None else interval)
    n_rays = pp.shape[0] * dd.shape[0]
    I = np.zeros((pp.shape[0], dd.shape[0], wl.n_lambda), dtype=np.float64)
    cap = counts = records = ds = None
    if capture:
        cap, counts, records, ds = _capture(n_rays, sum(wl.dims[:wl.ndim]) + 16, 0, keep)
    n = lib().orc_plain_march(C.byref(g), C.byref(F), pp.shape[0], pp.ctypes.data, dd.shape[0], dd.ctypes.data,
                              None if ii is None else ii.ctypes.data, I.ctypes.data,
                              C.byref(cap) if cap is not None else None, n_threads)
    if n < 0:
        raise RuntimeError("oracle plain march failed")
    return MarchResult(I=I, segments=int(n), counts=counts, records=records, ds=ds)


def velocity_bin_report(wl, factor=2.0, n_vbins=None):
    """bin spacing of the per-voxel velocity grid [-|v|, |v|] against the thermal width of
    each line, over the voxels of active bricks: (max ratio per line, voxels with ratio > factor per line)."""
    n = wl.n_vbins if n_vbins is None else n_vbins
    act = np.repeat(brick_active(wl).reshape(grid_shape_bricks(wl)), wl.brick, axis=-1)
    for ax in range(wl.ndim - 1):
        act = np.repeat(act, wl.brick, axis=ax)
    act = act.reshape(-1)
    V = np.sqrt((wl.vel.astype(np.float64) ** 2).sum(axis=1)).astype(np.float32).astype(np.float64)
    spacing = 2.0 * V / float(n - 1)
    mx, over = [], []
    for l in range(wl.n_lines):
        ratio = (spacing * wl.inv_dlamD[l].astype(np.float64) * float(wl.lambda0[l]) / float(np.float32(wl.c_light)))
        ratio = ratio.astype(np.float32)[act]
        mx.append(float(ratio.max()) if ratio.size else 0.0)
        over.append(int((ratio > np.float32(factor)).sum()))
    return np.asarray(mx, dtype=np.float32), np.asarray(over, dtype=np.int64)


def grid_shape_bricks(wl):
    bd = wl.brick_dims
    return (bd[1], bd[0]) if wl.ndim == 2 else (bd[2], bd[1], bd[0])


def level_caps_paper(n_levels=4, first=6.0, factor=4.0):
    """Distance thresholds of the near-field MIP cap: the long-characteristics analogue of DexRT's per-cascade
    maximum MIP level [0,0,1,2,3,4] with interval ends 1.5 * 4^i voxels: level <= 0 for t < 6,
    <= 1 for t < 24, <= 2 for t < 96, <= 3 for t < 384, unrestricted beyond."""
    return np.asarray([first * factor ** i for i in range(n_levels)], dtype=np.float32)


def hdda_march(wl, M: OracleMips, probe_pos=None, dirs=None, i0=None, capture_batch=None, levels=None,
               n_threads=0, level_cap_t=None, sin_incl=None, interval=None) -> MarchResult:
    """(B) HDDA over the brick/level structure with the VLM mips (Algorithm 1).
    level_cap_t: ascending distance thresholds of the near-field MIP cap (T8), None = no cap."""
    keep = []
    g, F = _make_structs(wl, M, keep)
    if level_cap_t is not None:
        caps = np.asarray(level_cap_t, dtype=np.float32)
        assert caps.size <= 8 and (np.diff(caps) >= 0).all()
        g.n_caps = int(caps.size)
        for i, v in enumerate(caps):
            g.cap_t[i] = float(v)
    if F.variant == CLASSIC:
        F.variant = CAV
    pp, dd, ii = _rays(wl, probe_pos, dirs, i0)
    _set_sin_incl(g, wl, dd, sin_incl, keep)
    _set_interval(g, getattr(wl, "interval", None) if interval is None else interval)
    lv = np.ascontiguousarray(M.levels if levels is None else levels, dtype=np.int8)
    n_rays = pp.shape[0] * dd.shape[0]
    I = np.zeros((pp.shape[0], dd.shape[0], wl.n_lambda), dtype=np.float64)
    cap = counts = records = ds = None
    if capture_batch is not None:
        cap, counts, records, ds = _capture(n_rays, sum(wl.dims[:wl.ndim]) + 16, int(capture_batch), keep)
    n = lib().orc_hdda_march(C.byref(g), C.byref(F), lv.ctypes.data, pp.shape[0], pp.ctypes.data, dd.shape[0],
                             dd.ctypes.data, None if ii is None else ii.ctypes.data, I.ctypes.data,
                             C.byref(cap) if cap is not None else None, n_threads)
    if n < 0:
        raise RuntimeError("oracle HDDA march failed")
    return MarchResult(I=I, segments=int(n), counts=counts, records=records, ds=ds)


def mean_intensity(I, weights):
    """J(p, lambda) = sum_k w_k I(p, k, lambda)."""
    I = np.ascontiguousarray(I, dtype=np.float64)
    w = np.ascontiguousarray(weights, dtype=np.float32)
    J = np.zeros((I.shape[0], I.shape[2]), dtype=np.float64)
    lib().orc_mean_intensity(I.shape[0], I.shape[1], I.shape[2], w.ctypes.data, I.ctypes.data, J.ctypes.data)
    return J


def unpack_record(rec):
    rec = np.asarray(rec, dtype=np.uint64)
    lvl = (rec >> np.uint64(56)).astype(np.int64)
    z = ((rec >> np.uint64(36)) & np.uint64(0x3FFFF)).astype(np.int64)
    y = ((rec >> np.uint64(18)) & np.uint64(0x3FFFF)).astype(np.int64)
    x = (rec & np.uint64(0x3FFFF)).astype(np.int64)
    return lvl, x, y, z


# --------------------------------------------------------------------------------------
# (C) brute-force geometry for tiny grids: slab intersection of the ray with every cell of the
# adapted grid, in fp64, sorted by entry distance -- independent of any DDA ("exact
# path length of the ray in each voxel").
# --------------------------------------------------------------------------------------

def brute_force_segments(wl, levels_row, probe, omega, min_len=0.0):
    nd, B = wl.ndim, wl.brick
    o = np.asarray(probe, dtype=np.float32).astype(np.float64)
    d = -np.asarray(omega, dtype=np.float32).astype(np.float64)
    bd = wl.brick_dims
    out = []
    for bi in range(wl.n_bricks):
        m = int(levels_row[bi])
        if m < 0:
            continue
        bx = bi % bd[0]
        by = (bi // bd[0]) % bd[1]
        bz = bi // (bd[0] * bd[1])
        size = 1 << m
        ncell = B // size
        rng_z = range(ncell) if nd == 3 else range(1)
        for cz in rng_z:
            for cy in range(ncell):
                for cx in range(ncell):
                    lo = np.array([bx * B + cx * size, by * B + cy * size, bz * B + cz * size][:nd], dtype=np.float64)
                    hi = lo + size
                    t0, t1 = 0.0, np.inf
                    hit = True
                    for a in range(nd):
                        if d[a] == 0.0:
                            if not (lo[a] <= o[a] < hi[a]):
                                hit = False
                                break
                        else:
                            ta, tb = (lo[a] - o[a]) / d[a], (hi[a] - o[a]) / d[a]
                            if ta > tb:
                                ta, tb = tb, ta
                            t0, t1 = max(t0, ta), min(t1, tb)
                    if hit and t1 - t0 > min_len:
                        cc = [int(lo[a]) >> m for a in range(nd)] + ([0] if nd == 2 else [])
                        out.append((t0, m, cc[0], cc[1], cc[2], t1 - t0))
    out.sort(key=lambda r: r[0])
    return out


# --------------------------------------------------------------------------------------
# Single-direction VLM (T11)
# --------------------------------------------------------------------------------------
def direction_fields(wl, omega, sin_incl=None):
    """Emissivity and opacity of an anisotropic medium as seen along ONE direction omega, at full resolution: the
    Classic formula (eqs. 10-20: background + sum over the batch's active lines of the Doppler-shifted Voigt profile)
    with v_proj = v . omega per voxel (times sin_incl for a 2.5D ray, T9), evaluated in fp64 and rounded
    once to fp32.  These are "a grid of emissivity and opacity given a single direction" to which the plain VLM method
    applies.  Voxels of unpopulated bricks are 0.  Returns (eta, chi), fp32 [nvox][n_lambda]."""
    nd, W, nl = wl.ndim, wl.lambda_batch, wl.n_lambda
    g0 = grid_shape(wl, 0)
    nL = wl.n_lines
    es, cs = wl.eta_star0.reshape((nL,) + g0), wl.chi_star0.reshape((nL,) + g0)
    a0, inv = wl.a0.reshape((nL,) + g0), wl.inv_dlamD.reshape((nL,) + g0)
    v0 = _to_grid(wl, wl.vel, 0, (nd,))
    om = np.asarray(omega, dtype=np.float32).astype(np.float64)
    vproj = np.zeros(g0, dtype=np.float64)
    for a in range(nd):
        vproj = vproj + v0[..., a].astype(np.float64) * om[a]
    if sin_incl is not None:
        vproj = vproj * float(np.float32(sin_incl))
    bg_e, bg_c = _to_grid(wl, wl.eta_bg, 0, (nl,)), _to_grid(wl, wl.chi_bg, 0, (nl,))
    eta = np.zeros(g0 + (nl,), dtype=np.float32)
    chi = np.zeros(g0 + (nl,), dtype=np.float32)
    for b in range(wl.n_batch):
        lines = [int(l) for l in wl.active_lines[b] if l >= 0]
        idx = np.arange(b * W, (b + 1) * W)
        ee, cc = _line_sum(wl, idx, lines, es, cs, a0, inv, {l: vproj for l in lines}, bg_e[..., idx], bg_c[..., idx])
        eta[..., idx] = ee.astype(np.float32)
        chi[..., idx] = cc.astype(np.float32)
    # voxels of unpopulated bricks carry nothing
    B = wl.brick
    act_b = brick_active(wl)
    bd = tuple(s // B for s in g0)
    vox_act = act_b.reshape(bd)
    for ax in range(nd):
        vox_act = np.repeat(vox_act, B, axis=ax)
    eta[~vox_act] = 0.0
    chi[~vox_act] = 0.0
    return eta.reshape(-1, nl), chi.reshape(-1, nl)


def single_direction_workload(wl, k):
    """The static (ISO) workload direction k of an anisotropic workload defines: its direction fields, that one ray
    direction with its quadrature weight and boundary intensity; thresholds, metric and max_level as wl's."""
    import copy
    s = copy.copy(wl)
    si = getattr(wl, "sin_incl", None)
    s.eta, s.chi = direction_fields(wl, wl.dirs[k], None if si is None else si[k])
    s.variant = ISO
    s.dirs = np.ascontiguousarray(wl.dirs[k:k + 1])
    s.weights = np.ascontiguousarray(wl.weights[k:k + 1])
    s.i0 = None if wl.i0 is None else np.ascontiguousarray(wl.i0[k:k + 1])
    s.sin_incl = None if si is None else np.ascontiguousarray(si[k:k + 1])
    return s


def single_direction_solve(wl, level_cap_t=None, n_threads=0):
    """for each quadrature direction, VLM on that direction's fields, HDDA march of that direction's
    rays; J = sum_k w_k I_k.  Returns (J fp64 [n_probes][n_lambda], levels int8
    [n_dirs][n_batch][n_bricks], emitted segments)."""
    n_dirs = wl.dirs.shape[0]
    I = np.zeros((wl.probe_pos.shape[0], n_dirs, wl.n_lambda), dtype=np.float64)
    levels, segs = [], 0
    for k in range(n_dirs):
        s = single_direction_workload(wl, k)
        M = build_mips(s, variant=ISO)
        r = hdda_march(s, M, level_cap_t=level_cap_t, n_threads=n_threads)
        I[:, k, :] = r.I[:, 0, :]
        levels.append(M.levels)
        segs += r.segments
    return mean_intensity(I, wl.weights), np.stack(levels), segs
