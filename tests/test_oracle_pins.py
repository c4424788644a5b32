"""Pins for the CPU oracle: closed forms, paper values, invariants, brute force.

None of these compares the oracle with itself through the same formula: every expected value is a
closed form typed here, a value printed in the paper (tests/golden), an independent geometric
computation, a library routine (scipy.special.wofz) or a second, differently structured
implementation.
"""
import math
import os

import numpy as np
import pytest

from oracle import oracle as orc
from workloads import make
from workloads.gen import dirs_2d, dirs_fibonacci, METRIC_RELVAR
from _util import (fig5_levels, iso_workload, max_rel, path_to_boundary, random_unit_dirs, unit_dirs_2d)

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ------------------------------------------------------------------ P1: homogeneous slab
@pytest.mark.parametrize("ndim", [2, 3])
def test_p1_homogeneous_slab_any_level(ndim):
    """with homogeneous parameters the averaged formulation is equivalent; any ray of
    length L through uniform chi, S gives I = I0 e^{-chi h L} + S (1 - e^{-chi h L}) whatever the
    cells and levels crossed."""
    rng = np.random.default_rng(11)
    brick = 16 if ndim == 2 else 8
    dims = (64, 48) if ndim == 2 else (24, 16, 32)
    chi0, S0, h = 0.037, 1.7, 1.3
    shape = dims[::-1]
    probes = rng.uniform(0.01, 0.99, size=(40, ndim)) * np.array(dims)
    dirs = random_unit_dirs(12, ndim, rng)
    i0 = rng.uniform(0.0, 3.0, size=(dirs.shape[0], 8))
    wl = iso_workload(dims, brick, np.full(shape, chi0 * S0), np.full(shape, chi0), probes, dirs, h=h,
                      max_level=int(math.log2(brick)), i0=i0)
    M = orc.build_mips(wl)
    nbr = wl.n_bricks
    lv = rng.integers(0, int(math.log2(brick)) + 1, size=(1, nbr)).astype(np.int8)   # arbitrary levels
    A = orc.plain_march(wl)
    B = orc.hdda_march(wl, M, levels=lv)
    chi32, eta32 = float(np.float32(chi0)), float(np.float32(chi0 * S0))
    for p in range(probes.shape[0]):
        for k in range(dirs.shape[0]):
            L = path_to_boundary(wl.probe_pos[p], wl.dirs[k], dims)
            att = math.exp(-chi32 * h * L)
            want = wl.i0[k, 0] * att + (eta32 / chi32) * (1.0 - att)
            assert abs(A.I[p, k, 0] - want) <= 3e-6 * abs(want)     # fp32 plane times: ~1e-6 in L
            assert abs(B.I[p, k, 0] - want) <= 3e-6 * abs(want)


def test_p1_table1_average_column():
    """Table 1: averaged eta = 1.2, chi = 0.8 over a corner-to-corner path sqrt(5)
    prints 1.25 in the 'Average' column of ray gamma."""
    rows = {}
    with open(os.path.join(GOLDEN, "table1.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            name, true, avg = line.split()
            rows[name] = (float(true), float(avg))
    eta_avg = (2 + 2 + 0.4 + 0.4) / 4
    chi_avg = (0.2 + 0.2 + 1.4 + 1.4) / 4
    got = orc.segment(0.0, eta_avg, chi_avg, math.sqrt(5.0))
    assert abs(got - 1.2492727) < 5e-7
    assert round(got, 2) == rows["gamma"][1]
    # the same through the march: 2x1 block of the averaged medium, ray along the diagonal
    th = math.atan2(1.0, 2.0)
    wl = iso_workload((2, 2), 2, np.full((2, 2), eta_avg), np.full((2, 2), chi_avg),
                      probes=[[np.nextafter(np.float32(2.0), np.float32(0)), np.nextafter(np.float32(1.0), np.float32(0))]],
                      dirs=unit_dirs_2d([th]))
    A = orc.plain_march(wl)
    assert abs(A.I[0, 0, 0] - 1.2492727) < 2e-6


# ------------------------------------------------------------------ P2: order of accumulation
def test_p2_order_dependence_table1_coefficients():
    """opposed rays through the same voxels differ.  Unit paths through a light
    (eta 2, chi .2) and a dark (eta .4, chi 1.4) voxel: hand-computed 0.6622625 / 1.9889308."""
    light = (2.0, 0.2)
    dark = (0.4, 1.4)
    I_ld = (light[0] / light[1]) * (1 - math.exp(-light[1]))
    I_ld = I_ld * math.exp(-dark[1]) + (dark[0] / dark[1]) * (1 - math.exp(-dark[1]))
    I_dl = (dark[0] / dark[1]) * (1 - math.exp(-dark[1]))
    I_dl = I_dl * math.exp(-light[1]) + (light[0] / light[1]) * (1 - math.exp(-light[1]))
    assert abs(I_ld - 0.6622625) < 1e-7 and abs(I_dl - 1.9889308) < 1e-7
    eta = np.array([[2.0, 0.4], [2.0, 0.4]])
    chi = np.array([[0.2, 1.4], [0.2, 1.4]])
    eps = 2.0 ** -20
    # radiation propagating +x ends in the dark voxel (light -> dark); propagating -x the reverse
    wl = iso_workload((2, 2), 2, eta, chi, probes=[[2.0 - eps, 0.5], [eps, 0.5]], dirs=[[1.0, 0.0], [-1.0, 0.0]])
    for res in (orc.plain_march(wl), orc.hdda_march(wl, orc.build_mips(wl))):
        assert abs(res.I[0, 0, 0] - 0.6622625) < 3e-6
        assert abs(res.I[1, 1, 0] - 1.9889308) < 3e-6
        assert res.I[0, 0, 0] < res.I[1, 1, 0]


# ------------------------------------------------------------------ P3: chi = 0 handling, thin limit
def test_p3_transparent_and_thin():
    """Zero-opacity voxels are transparent; for small chi ds the RTE is linear:
    I ~= sum eta h ds."""
    rng = np.random.default_rng(5)
    dims = (32, 32)
    eta = np.zeros(dims[::-1])
    chi = np.zeros(dims[::-1])
    eta[8:24, 8:24] = 1.0
    chi[8:24, 8:24] = 0.5
    probes = rng.uniform(1, 31, size=(30, 2))
    dirs = random_unit_dirs(8, 2, rng)
    i0 = np.full((8, 8), 0.7)
    wl = iso_workload(dims, 16, eta, chi, probes, dirs, i0=i0)
    A = orc.plain_march(wl, capture=True)
    # independent expectation: only the opaque square matters; its chord length from the capture
    for r in range(A.counts.shape[0]):
        n = A.counts[r]
        lvl, x, y, z = orc.unpack_record(A.records[r, :n])
        inside = (x >= 8) & (x < 24) & (y >= 8) & (y < 24)
        # segments are listed probe-outward: material in front of the square (towards the probe) is empty
        L = float(A.ds[r, :n][inside].astype(np.float64).sum())
        want = float(np.float32(0.7)) * math.exp(-0.5 * L) + 2.0 * (1 - math.exp(-0.5 * L))
        p, k = divmod(r, 8)
        assert abs(A.I[p, k, 0] - want) < 1e-12 + 1e-12 * want
    # pure emitter (chi = 0): I = I0 + eta h L exactly; thin medium: first-order
    wl2 = iso_workload(dims, 16, np.full(dims[::-1], 0.25), np.zeros(dims[::-1]), probes, dirs, h=2.0)
    A2 = orc.plain_march(wl2)
    wl3 = iso_workload(dims, 16, np.full(dims[::-1], 0.25), np.full(dims[::-1], 1e-9), probes, dirs, h=2.0)
    A3 = orc.plain_march(wl3)
    for p in range(30):
        for k in range(8):
            L = path_to_boundary(wl2.probe_pos[p], wl2.dirs[k], dims)
            assert abs(A2.I[p, k, 0] - 0.25 * 2.0 * L) < 3e-6 * 0.5 * L
            assert abs(A3.I[p, k, 0] - A2.I[p, k, 0]) < 1e-6 * A2.I[p, k, 0]


# ------------------------------------------------------------------ P4: J
def test_p4_mean_intensity():
    """J = sum_k w_k I_k.  Optically thick uniform medium: I -> S for every direction,
    so J -> S sum(w); and a hand example with unequal weights."""
    dims = (32, 32)
    wl = iso_workload(dims, 16, np.full(dims[::-1], 30.0 * 2.5), np.full(dims[::-1], 30.0), probes=[[16.5, 16.5]],
                      dirs=dirs_2d(16)[0])
    A = orc.plain_march(wl)
    J = orc.mean_intensity(A.I, wl.weights)
    assert abs(J[0, 0] - 2.5) < 1e-9
    I = np.arange(2 * 3 * 2, dtype=np.float64).reshape(2, 3, 2)
    w = np.array([0.5, 0.25, 0.125], dtype=np.float32)
    J = orc.mean_intensity(I, w)
    assert np.allclose(J, [[0 * .5 + 2 * .25 + 4 * .125, 1 * .5 + 3 * .25 + 5 * .125],
                           [6 * .5 + 8 * .25 + 10 * .125, 7 * .5 + 9 * .25 + 11 * .125]], rtol=0, atol=1e-15)


# ------------------------------------------------------------------ P5/P6: HDDA == plain DDA
def _lists_equal_filtered(wl, A, B):
    act_b = orc.brick_active(wl)
    bd = wl.brick_dims
    bad = 0
    for r in range(A.counts.shape[0]):
        na = A.counts[r]
        recA, dsA = A.records[r, :na], A.ds[r, :na]
        lvl, x, y, z = orc.unpack_record(recA)
        b = ((z // wl.brick) * bd[1] + y // wl.brick) * bd[0] + x // wl.brick
        keep = act_b[b]
        nb_ = B.counts[r]
        if keep.sum() != nb_ or not np.array_equal(recA[keep], B.records[r, :nb_]) or \
                not np.array_equal(dsA[keep].view(np.uint32), B.ds[r, :nb_].view(np.uint32)):
            bad += 1
    return bad


def test_p5_threshold_zero_reproduces_plain_march():
    """V7 / north_star: VLM threshold 0 and all bricks occupied => level 0 everywhere => the HDDA
    visit list and intensities are those of the plain march, bit for bit."""
    wl = make("C1", n=32, n_dirs=8)
    d0, _ = dirs_2d(8, phase=0.0)      # axis-aligned and exact diagonals too
    wl.dirs = np.concatenate([wl.dirs, d0]).astype(np.float32)
    wl.weights = np.full(16, 1 / 16, dtype=np.float32)
    M = orc.build_mips(wl, max_level=3, thr_eta=0.0, thr_chi=0.0)
    assert (M.levels == 0).all()
    A = orc.plain_march(wl, capture=True)
    B = orc.hdda_march(wl, M, capture_batch=0)
    assert _lists_equal_filtered(wl, A, B) == 0
    assert np.array_equal(A.I, B.I)


@pytest.mark.parametrize("ndim", [2, 3])
def test_p6_brick_skipping_equals_filtered_plain_list(ndim):
    """north_star: the HDDA voxel-visit list equals the plain DDA's non-empty visits, bitwise incl. ds."""
    if ndim == 2:
        wl = make("C2", n=128, n_dirs=12, n_probes=200)
        extra, _ = dirs_2d(8, phase=0.0)
        rng = np.random.default_rng(3)
        wl.probe_pos = np.concatenate([wl.probe_pos, rng.uniform(0, 128, size=(50, 2)).astype(np.float32)])
    else:
        wl = make("C5", n=32, n_dirs=12, n_probes=150)
        wl.variant = 0
        wl.eta, wl.chi = wl.eta_bg, wl.chi_bg
        extra = np.array([[1, 0, 0], [0, -1, 0], [0, 0, 1], [1, 1, 0], [1, 1, 1], [-1, 1, -1]], dtype=np.float64)
        extra = (extra / np.linalg.norm(extra, axis=1, keepdims=True)).astype(np.float32)
    wl.dirs = np.concatenate([wl.dirs, extra]).astype(np.float32)
    wl.weights = np.full(len(wl.dirs), 1.0 / len(wl.dirs), dtype=np.float32)
    M0 = orc.build_mips(wl, max_level=0, variant=0)
    assert (M0.levels < 0).any() and (M0.levels == 0).any()
    A = orc.plain_march(wl, M0, capture=True)
    B = orc.hdda_march(wl, M0, capture_batch=0)
    assert _lists_equal_filtered(wl, A, B) == 0
    assert np.array_equal(A.I, B.I)
    assert B.segments < A.segments


# ------------------------------------------------------------------ P7: mips + HDDA together
def test_p7_hdda_equals_plain_march_over_upsampled_field():
    """Segments with equal eta, chi compose exactly, so VLM+HDDA must equal the plain march over the
    field in which every voxel carries its cell's mip value (agreement to fp32 ds rounding)."""
    wl = make("C2", n=128, n_dirs=16, n_probes=300)
    M = orc.build_mips(wl, thr_eta=0.05, thr_chi=0.05)
    assert len(np.unique(M.levels)) >= 3
    B = orc.hdda_march(wl, M)
    # upsample: per batch, per brick, take the level-m chain repeated 2^m times
    n, b, W = 128, wl.brick, wl.lambda_batch
    eta_up = np.zeros((n, n, wl.n_lambda), dtype=np.float32)
    chi_up = np.zeros_like(eta_up)
    nbx = n // b
    for bt in range(wl.n_batch):
        sl = slice(bt * W, (bt + 1) * W)
        for bi in range(wl.n_bricks):
            m = int(M.levels[bt, bi])
            if m < 0:
                continue
            by, bx = divmod(bi, nbx)
            cb = b >> m
            for name, up in (("eta", eta_up), ("chi", chi_up)):
                src = getattr(M, name)[m][by * cb:(by + 1) * cb, bx * cb:(bx + 1) * cb, sl]
                up[by * b:(by + 1) * b, bx * b:(bx + 1) * b, sl] = np.repeat(np.repeat(src, 1 << m, axis=0), 1 << m, axis=1)
    wl_up = iso_workload((n, n), b, eta_up, chi_up, wl.probe_pos, wl.dirs, active=wl.active)
    A = orc.plain_march(wl_up)
    assert max_rel(B.I, A.I) < 2e-6


# ------------------------------------------------------------------ P8: brute-force geometry
def _check_against_brute_force(wl, levels_row, M, min_len=2e-3):
    B = orc.hdda_march(wl, M, levels=levels_row[None, :].repeat(wl.n_batch, axis=0), capture_batch=0)
    nd = wl.dirs.shape[0]
    for r in range(B.counts.shape[0]):
        p, k = divmod(r, nd)
        bf = orc.brute_force_segments(wl, levels_row, wl.probe_pos[p], wl.dirs[k], min_len=min_len)
        n = B.counts[r]
        lvl, x, y, z = orc.unpack_record(B.records[r, :n])
        ds = B.ds[r, :n].astype(np.float64)
        keep = ds > min_len
        got = list(zip(lvl[keep], x[keep], y[keep], z[keep]))
        want = [(s[1], s[2], s[3], s[4]) for s in bf]
        assert got == want, (r, got[:6], want[:6])
        assert np.allclose(ds[keep], [s[5] for s in bf], rtol=0, atol=3e-5)
        tot_bf = sum(s[5] for s in orc.brute_force_segments(wl, levels_row, wl.probe_pos[p], wl.dirs[k]))
        assert abs(ds.sum() - tot_bf) < 1e-4


def test_p8_fig5_fixture_brute_force():
    """Fig. 5: 32x32, 4x4 blocks of 8x8 with the listed block states; HDDA must give the
    geometric ray-cell intersections ("exact path length of the ray in each voxel")."""
    rng = np.random.default_rng(8)
    lv = fig5_levels()
    probes = np.concatenate([rng.uniform(0, 32, size=(12, 2)), [[16.5, 16.5], [0.5, 31.5], [20.25, 11.75]]])
    dirs = np.concatenate([random_unit_dirs(9, 2, rng), unit_dirs_2d([0.0, math.pi / 2, math.pi / 4, math.pi, 1.25 * math.pi])])
    f = rng.uniform(0.5, 1.5, size=(32, 32))
    wl = iso_workload((32, 32), 8, f, f, probes, dirs, max_level=3)
    M = orc.build_mips(wl, max_level=3)
    _check_against_brute_force(wl, lv, M)


def test_p8_random_3d_brute_force():
    rng = np.random.default_rng(9)
    lv = rng.integers(-1, 4, size=64).astype(np.int8)       # 4x4x4 bricks of 8^3, levels -1..3
    probes = rng.uniform(0, 32, size=(6, 3))
    dirs = np.concatenate([random_unit_dirs(6, 3, rng), [[0, 0, 1.0], [0.6, 0.8, 0.0]]])
    f = rng.uniform(0.5, 1.5, size=(32, 32, 32))
    wl = iso_workload((32, 32, 32), 8, f, f, probes, dirs, max_level=3)
    M = orc.build_mips(wl, max_level=3)
    _check_against_brute_force(wl, lv, M)


# ------------------------------------------------------------------ P9: pyramid sizes and packing
def test_p9_pyramid_sizes_and_packing():
    """PAPER.md:109 (1.33x / 1.14x), :142 (first two MIPs hold 94 % of 2D storage), :162 (3 bits per
    16-block state, 21 per 64-bit word, 49 words = 392 B for 512^2), :132-138 (fractions sum to 1)."""
    wl = make("C2", n=128, n_dirs=4, n_probes=4)
    M = orc.build_mips(wl, max_level=4, thr_eta=1.0, thr_chi=1.0)
    sizes = [a.size for a in M.eta]
    assert abs(sum(sizes[:4]) / sizes[0] - 1.328125) < 1e-12
    assert abs(sum(sizes) / sizes[0] - (1 + 1 / 4 + 1 / 16 + 1 / 64 + 1 / 256)) < 1e-12
    assert abs((sizes[0] + sizes[1]) / (sizes[0] * 4 / 3) - 0.9375) < 1e-12     # "94 %"
    assert abs(sum(8.0 ** -m for m in range(3)) - 1.140625) < 1e-15
    words = orc.pack_levels(np.zeros(1024, dtype=np.int8), 4)                   # 512^2 / 16^2 = 1024 blocks
    assert words.shape[0] == 49 and words.nbytes == 392
    lv = np.random.default_rng(1).integers(-1, 5, size=1024).astype(np.int8)
    w = orc.pack_levels(lv, 4)
    un = np.array([((int(w[i // 21]) >> ((i % 21) * 3)) & 7) - 1 for i in range(1024)])
    assert np.array_equal(un, lv)
    # level histogram area fractions sum to 1 (Table 2 rows)
    for b in range(wl.n_batch):
        hist = np.bincount(M.levels[b] + 1, minlength=6)
        assert hist.sum() == wl.n_bricks


# ------------------------------------------------------------------ P10: level selection
def _levels_by_loops(wl, max_level, metric, thr, tau_gate):
    """Second, differently structured implementation of V1-V5 for ISO: per brick, per wavelength,
    python floats (fp64), explicit loops.  2D only."""
    n, B, W, h = wl.dims[0], wl.brick, wl.lambda_batch, float(wl.voxel_size)
    thr, tau_gate = float(np.float32(thr)), float(np.float32(tau_gate))     # fp32 at the C ABI
    eta = wl.eta.reshape(n, n, wl.n_lambda)
    chi = wl.chi.reshape(n, n, wl.n_lambda)
    act = wl.active.reshape(n, n)
    nb = n // B
    out = np.zeros((wl.n_batch, nb * nb), dtype=np.int8)

    def stat(vals):
        if all(v == vals[0] for v in vals):
            return 0.0
        if metric == orc.IOD_LOG:
            if any(v <= 0 for v in vals):
                return math.inf
            X = [math.log(v * h) for v in vals]
        else:
            X = list(vals)
        mean = (((X[0] + X[1]) + X[2]) + X[3]) / 4
        var = (((X[0] - mean) ** 2 + (X[1] - mean) ** 2) + (X[2] - mean) ** 2 + (X[3] - mean) ** 2) / 4
        if metric == orc.IOD_LOG:
            return abs(var / mean) if mean != 0 else math.inf
        return var / (mean * mean) if mean != 0 else math.inf

    for by in range(nb):
        for bx in range(nb):
            bi = by * nb + bx
            if not act[by * B:(by + 1) * B, bx * B:(bx + 1) * B].any():
                out[:, bi] = -1
                continue
            for bt in range(wl.n_batch):
                level = 0
                ce = [eta[by * B:(by + 1) * B, bx * B:(bx + 1) * B, bt * W:(bt + 1) * W].astype(np.float64)]
                cc = [chi[by * B:(by + 1) * B, bx * B:(bx + 1) * B, bt * W:(bt + 1) * W].astype(np.float64)]
                for m in range(1, max_level + 1):
                    pe, pc = ce[-1], cc[-1]
                    s = pe.shape[0] // 2
                    ne = np.zeros((s, s, W))
                    nc = np.zeros((s, s, W))
                    ok = True
                    for j in range(s):
                        for i in range(s):
                            for l in range(W):
                                ve = [float(pe[2 * j, 2 * i, l]), float(pe[2 * j, 2 * i + 1, l]),
                                      float(pe[2 * j + 1, 2 * i, l]), float(pe[2 * j + 1, 2 * i + 1, l])]
                                vc = [float(pc[2 * j, 2 * i, l]), float(pc[2 * j, 2 * i + 1, l]),
                                      float(pc[2 * j + 1, 2 * i, l]), float(pc[2 * j + 1, 2 * i + 1, l])]
                                ne[j, i, l] = np.float32((((ve[0] + ve[1]) + ve[2]) + ve[3]) * 0.25)
                                nc[j, i, l] = np.float32((((vc[0] + vc[1]) + vc[2]) + vc[3]) * 0.25)
                                passed = stat(ve) < thr and stat(vc) < thr
                                if tau_gate >= 0 and ((((vc[0] + vc[1]) + vc[2]) + vc[3]) / 4) * h <= tau_gate:
                                    passed = True
                                ok = ok and passed
                    if not ok:
                        break
                    level = m
                    ce.append(ne)
                    cc.append(nc)
                out[bt, bi] = level
    return out


@pytest.mark.parametrize("metric,thr,gate", [(orc.RELVAR, 1e-2, -1.0), (orc.RELVAR, 0.2, -1.0),
                                             (orc.IOD_LOG, 1.0, 0.25), (orc.IOD_LOG, 0.05, -1.0)])
def test_p10_level_selection_second_implementation(metric, thr, gate):
    wl = make("C2", n=64, n_dirs=4, n_probes=4, n_lambda=16)
    M = orc.build_mips(wl, max_level=4, metric=metric, thr_eta=thr, thr_chi=thr, tau_gate=gate)
    ref = _levels_by_loops(wl, 4, metric, thr, gate)
    assert np.array_equal(M.levels, ref)


def test_p10_uniform_brick_and_hand_example_and_monotone():
    """Uniform brick: IoD = 0, passes for thr > 0, fails for thr = 0 (strict '<').
    Hand 2x2 example: values (1,1,3,3): mean 2, var 1, relvar 0.25; ln-values: IoD = |var/mean| of
    (0,0,ln3,ln3): var = (ln3/2)^2, mean = ln3/2 -> IoD = ln3/2 = 0.5493."""
    dims = (16, 16)
    u = np.full(dims, 0.3)
    wl = iso_workload(dims, 16, u, u, [[1.5, 1.5]], [[1.0, 0.0]], max_level=4)
    assert (orc.build_mips(wl, thr_eta=1e-9, thr_chi=1e-9).levels == 4).all()
    assert (orc.build_mips(wl, thr_eta=0.0, thr_chi=0.0).levels == 0).all()
    x = np.ones(dims)
    x[1::2, :] = 3.0                    # children of every level-1 cell: (1,1,3,3)
    wl = iso_workload(dims, 16, x, x, [[1.5, 1.5]], [[1.0, 0.0]], max_level=4)
    assert (orc.build_mips(wl, metric=orc.RELVAR, thr_eta=0.2501, thr_chi=0.2501).levels >= 1).all()
    assert (orc.build_mips(wl, metric=orc.RELVAR, thr_eta=0.2499, thr_chi=0.2499).levels == 0).all()
    assert (orc.build_mips(wl, metric=orc.IOD_LOG, thr_eta=0.5494, thr_chi=0.5494).levels >= 1).all()
    assert (orc.build_mips(wl, metric=orc.IOD_LOG, thr_eta=0.5492, thr_chi=0.5492).levels == 0).all()
    # gate: chi h = 2 on average; gate above it lets everything be averaged, whatever the variance
    assert (orc.build_mips(wl, metric=orc.RELVAR, thr_eta=0.0, thr_chi=0.0, tau_gate=2.0).levels == 4).all()
    assert (orc.build_mips(wl, metric=orc.RELVAR, thr_eta=0.0, thr_chi=0.0, tau_gate=1.99).levels == 0).all()
    # monotone in the threshold
    wl = make("C2", n=128, n_dirs=4, n_probes=4)
    prev = None
    for thr in (0.0, 1e-3, 1e-2, 1e-1, 1.0):
        lv = orc.build_mips(wl, max_level=4, thr_eta=thr, thr_chi=thr).levels
        if prev is not None:
            assert (lv >= prev).all()
        prev = lv


def test_v1_mip_values_are_correctly_rounded_means():
    rng = np.random.default_rng(2)
    a = np.exp(rng.standard_normal((8, 8, 3)) * 4).astype(np.float32)
    m = orc.mip_mean(a, 2)
    from fractions import Fraction
    for j in range(4):
        for i in range(4):
            for c in range(3):
                ex = sum(Fraction(float(a[2 * j + dy, 2 * i + dx, c])) for dy in (0, 1) for dx in (0, 1)) / 4
                assert float(m[j, i, c]) == float(np.float32(float(ex)))


# ------------------------------------------------------------------ P13: Voigt
def test_p13_voigt_against_wofz_and_normalisation():
    """HUM1WEI24 against scipy.special.wofz: <= 3e-7 relative at a = 0.01 inside the
    Weideman region, <= 7e-5 in Humlicek's region I (the approximation's own error);
    and the profile integrates to 1."""
    from scipy.special import wofz
    x = np.linspace(-40, 40, 16001)
    for a, tol_in in ((0.01, 3e-7), (0.1, 3e-8), (1.0, 2e-9)):
        H = orc.voigt_H(a, x)
        ref = wofz(x + 1j * a).real
        rel = np.abs(H - ref) / ref
        inner = np.abs(x) + a < 15.0
        assert rel[inner].max() < tol_in
        assert rel[~inner].max() < 7e-5
    xx = np.linspace(-2000, 2000, 2_000_001)
    H = orc.voigt_H(0.01, xx)
    integral = np.trapezoid(H, xx) / math.sqrt(math.pi)
    assert abs(integral + 2 * 0.01 / (math.pi * 2000) - 1.0) < 2e-6    # Lorentz tail beyond +-2000 added back
    assert abs(orc.voigt_H(0.0, 0.0) - 1.0) < 1e-9
    assert abs(orc.voigt_H(0.0, 1.5) - math.exp(-2.25)) < 1e-8


# ------------------------------------------------------------------ P11 / P12: anisotropic providers
def _aniso_small(name, **kw):
    wl = make(name, **kw)
    return wl


def test_p12_cav_level0_equals_classic_and_rest_frame_identity():
    """Cav at level 0 with per-voxel v is the Classic brute force; at v = 0 and
    lambda = lambda0 eqs. 18-20 are the identity and eq. 14 the static profile."""
    wl = make("C4", n=64, n_dirs=6, n_probes=40)
    Mc = orc.build_mips(wl, max_level=0)
    A = orc.plain_march(wl, variant=orc.CLASSIC)
    B = orc.hdda_march(wl, Mc)
    assert max_rel(B.I, A.I) < 1e-12
    e, c = orc.line_terms(500.0, 500.0, 3.0, 7.0, 0.01, 40.0, 0.0, 299792.458)
    phi0 = orc.voigt_H(0.01, 0.0) * 40.0 / math.sqrt(math.pi)
    assert abs(e - 3.0 * phi0) < 1e-15 * abs(e) + 1e-300 and abs(c - 7.0 * phi0) < 1e-15 * abs(c)
    # Doppler shift moves the line centre to lambda0 (1 - v.w/c) (eq. 14 and eq. 17)
    v = 20.0
    lam_c = 500.0 * (1 - v / 299792.458)
    e_c, _ = orc.line_terms(lam_c, 500.0, 1.0, 1.0, 0.01, 40.0, v, 299792.458)
    e_l, _ = orc.line_terms(lam_c - 0.01, 500.0, 1.0, 1.0, 0.01, 40.0, v, 299792.458)
    e_r, _ = orc.line_terms(lam_c + 0.01, 500.0, 1.0, 1.0, 0.01, 40.0, v, 299792.458)
    assert e_c > e_l and e_c > e_r


def test_p12_static_medium_is_isotropic():
    wl = make("C3", n=64, n_dirs=8, n_probes=30)
    wl.vel[:] = 0.0
    Mc = orc.build_mips(wl, max_level=0, variant=orc.CAV)
    A = orc.plain_march(wl, variant=orc.CLASSIC)
    # rest-frame fields computed once, marched as ISO
    lam = wl.lam.astype(np.float64)
    e, c = orc.line_terms(lam[None, :], 500.0, wl.eta_star0[0][:, None], wl.chi_star0[0][:, None],
                          wl.a0[0][:, None], wl.inv_dlamD[0][:, None], 0.0, wl.c_light)
    iso = iso_workload(wl.dims[:2], wl.brick, (wl.eta_bg + e).reshape(64, 64, -1), (wl.chi_bg + c).reshape(64, 64, -1),
                       wl.probe_pos, wl.dirs, active=wl.active)
    C_ = orc.plain_march(iso)
    assert max_rel(A.I, C_.I) < 3e-7        # iso fields are rounded to fp32 once


def test_p11_velinterp_static_nodes_and_convergence():
    """VelInterp: v = 0 => table interpolation returns the static field; exact at
    bin nodes; converges to Classic as n grows."""
    wl = make("C3", n=64, n_dirs=8, n_probes=40)
    A = orc.plain_march(wl, variant=orc.CLASSIC)
    errs = []
    for n in (8, 32, 128):
        wl.n_vbins = n
        Mv = orc.build_mips(wl, max_level=0, variant=orc.VELINTERP)
        B = orc.hdda_march(wl, Mv)
        errs.append(np.percentile(np.abs(B.I - A.I) / np.maximum(A.I, 1e-300), 99))
    assert errs[2] < errs[1] < errs[0] and errs[2] < 1e-2
    # exact at nodes: a direction parallel to v projects onto the last bin
    wl.n_vbins = 8
    Mv = orc.build_mips(wl, max_level=0, variant=orc.VELINTERP)
    nv = wl.nvox
    V = np.sqrt((wl.vel.astype(np.float64) ** 2).sum(-1))
    vox = int(np.argmax(V))
    lam = wl.lam.astype(np.float64)
    e, c = orc.line_terms(lam, 500.0, wl.eta_star0[0][vox], wl.chi_star0[0][vox], wl.a0[0][vox],
                          wl.inv_dlamD[0][vox], float(np.float32(V[vox])), wl.c_light)
    tab = Mv.vtab[0].reshape(nv, 8, wl.n_lambda, 2)[vox]
    assert np.allclose(tab[7, :, 0], (wl.eta_bg[vox] + e).astype(np.float32), rtol=2e-7)
    assert np.allclose(tab[7, :, 1], (wl.chi_bg[vox] + c).astype(np.float32), rtol=2e-7)
    # static medium: every bin equal => interpolation is the static value
    wl.vel[:] = 0.0
    Mv0 = orc.build_mips(wl, max_level=0, variant=orc.VELINTERP)
    B0 = orc.hdda_march(wl, Mv0)
    A0 = orc.plain_march(wl, variant=orc.CLASSIC)
    assert max_rel(B0.I, A0.I) < 3e-7


def test_aniso_mips_hdda_consistency():
    """With mips on, Cav/VelInterp levels are populated and the HDDA result stays close to Classic
    (sanity: accuracy is reported, not gated -- SURVEY.md 8(d))."""
    for name in ("C3", "C4"):
        wl = make(name, n=256, n_dirs=8, n_probes=40)
        M = orc.build_mips(wl)
        assert M.levels.max() >= 1 and (M.levels == -1).any()
        B = orc.hdda_march(wl, M)
        A = orc.plain_march(wl, variant=orc.CLASSIC)
        J_b = orc.mean_intensity(B.I, wl.weights)
        J_a = orc.mean_intensity(A.I, wl.weights)
        ok = J_a > 0
        rel = np.abs(J_b[ok] - J_a[ok]) / J_a[ok]
        assert np.percentile(rel, 90) < 0.2


# ------------------------------------------------------------------------------------------------
# T8: near-field MIP cap (PAPER.md:347-349 per-cascade caps [0,0,1,2,3,4])
# ------------------------------------------------------------------------------------------------
def _slab(lvl, cc, probe, omega):
    """fp64 slab-method (entry, exit) distances of the ray through cell `cc` of level `lvl` (independent of any DDA)."""
    o = np.asarray(probe, dtype=np.float32).astype(np.float64)
    d = -np.asarray(omega, dtype=np.float32).astype(np.float64)
    size = float(1 << lvl)
    t0, t1 = 0.0, np.inf
    for a in range(len(o)):
        lo, hi = cc[a] * size, (cc[a] + 1) * size
        if d[a] != 0.0:
            ta, tb = (lo - o[a]) / d[a], (hi - o[a]) / d[a]
            t0 = max(t0, min(ta, tb))
            t1 = min(t1, max(ta, tb))
    return t0, t1


def test_t8_level_cap_limits_and_geometry():
    """(i) no thresholds, or thresholds that are all passed at t = 0, change nothing; (ii) thresholds never reached
    give level 0 everywhere, i.e. bit for bit the march over a level-0 table; (iii) on the Fig. 5 fixture every visited
    cell has level min(brick level, #{thresholds <= distance at which the visit starts}) with the distances from an
    independent fp64 slab intersection, and the path lengths still add up to the ray's length inside non-empty bricks;
    (iv) a homogeneous medium is still exact."""
    wl = make("C2", n=128, n_dirs=8, n_probes=150)
    wl.thr_eta = wl.thr_chi = 0.05
    M = orc.build_mips(wl)
    assert M.levels.max() >= 2
    a = orc.hdda_march(wl, M, capture_batch=1)
    for caps in ([], [0.0, 0.0, 0.0]):
        b = orc.hdda_march(wl, M, capture_batch=1, level_cap_t=caps)
        assert np.array_equal(a.records, b.records) and np.array_equal(a.ds.view(np.uint32), b.ds.view(np.uint32))
        assert np.array_equal(a.I, b.I)
    M0 = orc.build_mips(wl, max_level=0)
    z = orc.hdda_march(wl, M0, capture_batch=1)
    c = orc.hdda_march(wl, M, capture_batch=1, level_cap_t=[1e9, 1e9, 1e9])
    assert np.array_equal(z.records, c.records) and np.array_equal(z.ds.view(np.uint32), c.ds.view(np.uint32))
    assert np.array_equal(z.I, c.I)
    # (iii) Fig. 5 fixture: 32x32, 4x4 blocks of 8x8, levels up to 3
    rng = np.random.default_rng(21)
    lv = fig5_levels()
    lv = np.where(lv >= 0, 3, -1).astype(np.int8)          # every populated block at the coarsest level
    probes = rng.uniform(0, 32, size=(60, 2))
    dirs = random_unit_dirs(12, 2, rng)
    f = np.full((32, 32, 8), 0.3)
    act = np.repeat(np.repeat((lv >= 0).reshape(4, 4), 8, axis=0), 8, axis=1)
    f[~act] = 0.0
    wl5 = iso_workload((32, 32), 8, f * 1.7, f, probes, dirs, active=act.astype(np.uint8), max_level=3)
    M5 = orc.build_mips(wl5, max_level=3)
    M5.levels = np.ascontiguousarray(lv[None, :])
    caps = np.array([3.0, 7.5, 16.0], dtype=np.float32)
    r = orc.hdda_march(wl5, M5, capture_batch=0, level_cap_t=caps)
    seen = set()
    n_dirs = dirs.shape[0]
    for ray in range(r.counts.shape[0]):
        p, k = divmod(ray, n_dirs)
        n = int(r.counts[ray])
        lvl, x, y, _ = orc.unpack_record(r.records[ray, :n])
        prev_out = 0.0
        for i in range(n):
            # a visit starts where the ray enters the cell, or -- when a threshold was passed inside a coarse cell that
            # had been crossed as finer cells so far -- where the previous visit ended
            t_in, t_out = _slab(int(lvl[i]), (int(x[i]), int(y[i])), wl5.probe_pos[p], wl5.dirs[k])
            te = max(t_in, prev_out)
            prev_out = t_out
            if np.min(np.abs(caps.astype(np.float64) - te)) < 1e-3:
                continue                                     # entry within rounding of a threshold
            assert int(lvl[i]) == min(3, int((caps <= te).sum())), (ray, i, te, int(lvl[i]))
            seen.add(int(lvl[i]))
        tot_bf = sum(s[5] for s in orc.brute_force_segments(wl5, lv, wl5.probe_pos[p], wl5.dirs[k]))
        assert abs(float(r.ds[ray, :n].astype(np.float64).sum()) - tot_bf) < 2e-4
    assert seen == {0, 1, 2, 3}
    # (iv) uniform chi, S: closed form for every ray regardless of the levels used
    chi0 = float(np.float32(0.3))
    S0 = float(np.float32(0.3 * 1.7)) / chi0
    for ray in range(r.counts.shape[0]):
        n = int(r.counts[ray])
        L = float(r.ds[ray, :n].astype(np.float64).sum())
        assert abs(r.I[ray // n_dirs, ray % n_dirs, 0] - S0 * (1.0 - math.exp(-chi0 * L))) < 1e-12


def test_c13_velocity_bin_spacing_report_hand_example():
    """PAPER.md:200 warning criterion on a hand-checkable field: |v| = 30 km/s everywhere, 8 bins -> spacing 60/7 km/s;
    thermal width c dlamD / lambda0 = 5 km/s in the left half, 3 km/s in the right half -> ratios 12/7 and 20/7:
    only the right half exceeds the paper's factor 2."""
    wl = make("C3", n=64, n_dirs=4, n_probes=4)
    wl.active[:] = 1
    wl.vel[:, 0], wl.vel[:, 1] = 18.0, 24.0
    vth = np.where(np.arange(64)[None, :] < 32, 5.0, 3.0) * np.ones((64, 1))
    wl.inv_dlamD[0] = (wl.c_light / (vth.ravel() * float(wl.lambda0[0]))).astype(np.float32)
    mx, over = orc.velocity_bin_report(wl, factor=2.0)
    assert abs(float(mx[0]) - 20.0 / 7.0) < 1e-5 and int(over[0]) == 64 * 32
    mx, over = orc.velocity_bin_report(wl, factor=1.5)
    assert int(over[0]) == 64 * 64
    mx16, over16 = orc.velocity_bin_report(wl, factor=2.0, n_vbins=16)      # twice the bins: nothing to warn about
    assert abs(float(mx16[0]) - 4.0 / 3.0) < 1e-5 and int(over16[0]) == 0


# ------------------------------------------------------------------------------------------------
# 2.5D rays (PAPER.md:347 Gauss-Radau quadrature in the inclination to the homogeneous axis)
# ------------------------------------------------------------------------------------------------
def test_25d_quadrature_and_inclined_rays():
    """(i) the Gauss-Radau rule has its fixed node at mu = 0, weights summing to 1, and is exact to degree 2n - 2;
    (ii) sin = 1 changes nothing; (iii) homogeneous medium: I = S (1 - exp(-chi h L / sin)) with L the in-plane length
    (PAPER.md:65); (iv) an inclined ray equals an in-plane ray through the atmosphere with voxel size h / sin and
    velocities v sin (Classic march, eq. 14), visit lists unchanged; (v) J of a thick uniform medium is S."""
    from workloads.gen import dirs_25d, gauss_radau_unit
    for n in (2, 3, 4, 6):
        mu, w = gauss_radau_unit(n)
        assert mu[0] == 0.0 and abs(w.sum() - 1.0) < 1e-14 and (np.diff(mu) > 0).all() and mu[-1] < 1.0
        for k in range(2 * n - 1):
            assert abs((w * mu ** k).sum() - 1.0 / (k + 1)) < 1e-13
        assert abs((w * mu ** (2 * n - 1)).sum() - 1.0 / (2 * n)) > 1e-8
    # (ii), (iii)
    rng = np.random.default_rng(3)
    chi0, S0 = 0.07, 1.3
    f = np.full((48, 48, 8), chi0)
    probes = rng.uniform(0, 48, size=(20, 2))
    dirs, wts, si = dirs_25d(6, 4)
    wl = iso_workload((48, 48), 16, f * S0, f, probes, dirs, weights=wts, max_level=2, thr=1.0, h=1.5)
    M = orc.build_mips(wl)
    a = orc.hdda_march(wl, M, capture_batch=0)
    b = orc.hdda_march(wl, M, capture_batch=0, sin_incl=np.ones(len(si), dtype=np.float32))
    assert np.array_equal(a.I, b.I) and np.array_equal(a.records, b.records)
    c = orc.hdda_march(wl, M, capture_batch=0, sin_incl=si)
    assert np.array_equal(a.records, c.records) and np.array_equal(a.ds, c.ds)
    chi32, S32 = float(np.float32(chi0)), float(np.float32(chi0 * S0)) / float(np.float32(chi0))
    for p in range(probes.shape[0]):
        for k in range(dirs.shape[0]):
            L = path_to_boundary(wl.probe_pos[p], wl.dirs[k], (48, 48))
            want = S32 * (1.0 - math.exp(-chi32 * 1.5 * L / float(si[k])))
            assert abs(c.I[p, k, 0] - want) < 2e-5 * want          # L from fp64 geometry, ds from fp32 plane times
    # (iv) Classic march with velocities: inclined == in-plane with h / sin and v sin, one direction at a time
    wv = make("C4", n=64, n_dirs=3, n_probes=12)
    s = np.float32(0.59375)                                         # exactly representable
    A = orc.plain_march(wv, variant=orc.CLASSIC, sin_incl=np.full(3, s, dtype=np.float32), capture=True)
    import copy
    w2 = copy.copy(wv)
    w2.voxel_size = float(np.float64(wv.voxel_size) / np.float64(s))
    w2.vel = (wv.vel.astype(np.float64) * float(s)).astype(np.float32)
    Bm = orc.plain_march(w2, variant=orc.CLASSIC, capture=True)
    assert np.array_equal(A.records, Bm.records)
    assert max_rel(A.I, Bm.I) < 5e-6                                 # v sin and h / sin are rounded to fp32 in w2
    plain = orc.plain_march(wv, variant=orc.CLASSIC)
    assert max_rel(A.I, plain.I) > 1e-2                              # and the inclination does matter
    # (v) thick uniform medium: J -> S for the full 2.5D quadrature
    f2 = np.full((32, 32, 8), 5.0)
    wt = iso_workload((32, 32), 16, f2 * 0.8, f2, [[16.5, 16.5]], dirs, weights=wts)
    r = orc.plain_march(wt, sin_incl=si)
    J = orc.mean_intensity(r.I, wt.weights)
    assert abs(J[0, 0] - 0.8) < 1e-6


# ------------------------------------------------------------------------------------------------
# T10: finite radiance intervals (Algorithm 1 HDDA(t1, t2))
# ------------------------------------------------------------------------------------------------
def test_t10_radiance_intervals_compose():
    """(i) an interval that covers the ray changes nothing; (ii) the formal solution composes over a split of the
    ray: I(0, inf) = I(0, t) + T(0, t) I(t, inf), with T(0, t) = e^-tau obtained from the same march with eta = 0 and
    unit incoming intensity (eq. 3); (iii) the visit list of an interval is a contiguous run of the full list with
    only its first and last path lengths shortened; (iv) homogeneous medium closed form on [t1, t2]."""
    wl = make("C2", n=128, n_dirs=8, n_probes=120)
    wl.thr_eta = wl.thr_chi = 0.05
    M = orc.build_mips(wl)
    full = orc.hdda_march(wl, M, capture_batch=0)
    same = orc.hdda_march(wl, M, capture_batch=0, interval=(0.0, 1.0e9))
    assert np.array_equal(full.I, same.I) and np.array_equal(full.records, same.records)
    assert np.array_equal(full.ds.view(np.uint32), same.ds.view(np.uint32))
    for tsplit in (3.25, 17.3, 61.0):
        a = orc.hdda_march(wl, M, capture_batch=0, interval=(0.0, tsplit))
        b = orc.hdda_march(wl, M, capture_batch=0, interval=(tsplit, 1.0e9))
        import copy
        w0 = copy.copy(wl)
        w0.eta = np.zeros_like(wl.eta)
        M0 = copy.copy(M)
        M0.wl = w0
        M0.eta = [np.zeros_like(e) for e in M.eta]
        one = np.ones((wl.dirs.shape[0], wl.n_lambda), dtype=np.float32)
        Ta = orc.hdda_march(w0, M0, i0=one, interval=(0.0, tsplit)).I
        assert (Ta <= 1.0).all() and (Ta > 0.0).all()
        assert max_rel(a.I + Ta * b.I, full.I) < 1e-12
        # (iii)
        for ray in range(full.counts.shape[0]):
            nf, na, nb = int(full.counts[ray]), int(a.counts[ray]), int(b.counts[ray])
            assert nf - 0 <= na + nb <= nf + 1                    # the cell that contains tsplit appears in both
            assert np.array_equal(a.records[ray, :na], full.records[ray, :na])
            assert np.array_equal(b.records[ray, :nb], full.records[ray, nf - nb:nf])
            if na > 1:
                assert np.array_equal(a.ds[ray, :na - 1], full.ds[ray, :na - 1])
            if nb > 1:
                assert np.array_equal(b.ds[ray, 1:nb], full.ds[ray, nf - nb + 1:nf])
            tot = float(a.ds[ray, :na].astype(np.float64).sum() + b.ds[ray, :nb].astype(np.float64).sum())
            assert abs(tot - float(full.ds[ray, :nf].astype(np.float64).sum())) < 2e-4
    # (iv)
    f = np.full((40, 40, 8), 0.11)
    rng = np.random.default_rng(2)
    probes = rng.uniform(0, 40, size=(15, 2))
    wh = iso_workload((40, 40), 8, f * 2.5, f, probes, dirs_2d(7)[0], max_level=2, thr=1.0, h=0.8)
    Mh = orc.build_mips(wh)
    t1, t2 = 2.5, 19.0
    r = orc.hdda_march(wh, Mh, interval=(t1, t2))
    chi32 = float(np.float32(0.11))
    S32 = float(np.float32(0.11 * 2.5)) / chi32
    for p in range(probes.shape[0]):
        for k in range(7):
            L = path_to_boundary(wh.probe_pos[p], wh.dirs[k], (40, 40))
            seg = max(0.0, min(L, t2) - t1)
            want = S32 * (1.0 - math.exp(-chi32 * 0.8 * seg))
            assert abs(r.I[p, k, 0] - want) < 2e-5 * max(want, 1e-3)


# ------------------------------------------------------------------------------------------------
# 8(f)-3: wavelength batches are independent (one level table per batch), which is what lets the
# rebuild pipeline build and solve the spectrum stage by stage
# ------------------------------------------------------------------------------------------------
def test_batches_are_independent_in_the_oracle():
    import copy
    wl = make("C2", n=128, n_dirs=6, n_probes=60)
    M = orc.build_mips(wl)
    full = orc.hdda_march(wl, M)
    assert len({M.levels[b].tobytes() for b in range(wl.n_batch)}) > 1      # the batches do differ (core vs wing)
    for b0, b1 in ((0, 1), (1, 3), (3, 4)):
        sub = copy.copy(wl)
        sl = slice(b0 * wl.lambda_batch, b1 * wl.lambda_batch)
        sub.eta = np.ascontiguousarray(wl.eta[..., sl])
        sub.chi = np.ascontiguousarray(wl.chi[..., sl])
        sub.n_lambda = (b1 - b0) * wl.lambda_batch
        Ms = orc.build_mips(sub)
        assert np.array_equal(Ms.levels, M.levels[b0:b1])
        r = orc.hdda_march(sub, Ms)
        assert np.array_equal(r.I, full.I[..., sl])


# ------------------------------------------------------------------------------------------------
# T11: single-direction VLM
# ------------------------------------------------------------------------------------------------
def test_t11_direction_fields_and_single_direction_solve():
    """(i) a direction field value against the textbook formula with scipy's Faddeeva function (not the oracle's
    HUM1WEI24): eta = eta_bg + (lam0/lam) eta*_0 H(a, x) / (sqrt(pi) dlamD), x from the projected velocity;
    (ii) v -> -v together with omega -> -omega leaves the fields unchanged, v = 0 makes them direction independent;
    (iii) with mips off the per-direction static marches reproduce the Classic march (fields rounded to fp32 once);
    (iv) with mips on, each direction's level table is the ISO table of that direction's fields, differs between
    directions, and J stays within the VLM error of the exact Classic J."""
    from scipy.special import wofz
    wl = make("C4", n=64, n_dirs=6, n_probes=50)
    nl = wl.n_lambda
    om = wl.dirs[2]
    eta, chi = orc.direction_fields(wl, om)
    act = orc.brick_active(wl)
    rng = np.random.default_rng(5)
    vox_ok = np.flatnonzero(wl.active.ravel() != 0)
    for v in rng.choice(vox_ok, size=40, replace=False):
        for j in rng.choice(nl, size=6, replace=False):
            b = j // wl.lambda_batch
            lam = float(wl.lam[j])
            vproj = sum(float(wl.vel[v, a]) * float(om[a]) for a in range(wl.ndim))
            e, c = float(wl.eta_bg[v, j]), float(wl.chi_bg[v, j])
            for l in [int(q) for q in wl.active_lines[b] if q >= 0]:
                lam0, inv = float(wl.lambda0[l]), float(wl.inv_dlamD[l][v])
                x = (lam - lam0 + vproj / wl.c_light * lam0) * inv
                a = (lam / lam0) ** 2 * float(wl.a0[l][v])
                phi = wofz(x + 1j * a).real * inv / math.sqrt(math.pi)
                e += lam0 / lam * float(wl.eta_star0[l][v]) * phi
                c += lam0 / lam * float(wl.chi_star0[l][v]) * phi
            # HUM1WEI24's own error is ~1e-11 absolute in H, i.e. up to ~1e-6 relative in the far wings (p13)
            assert abs(eta[v, j] - e) <= 3e-6 * e and abs(chi[v, j] - c) <= 3e-6 * c
    # (ii)
    import copy
    wm = copy.copy(wl)
    wm.vel = -wl.vel
    e2, c2 = orc.direction_fields(wm, -om)
    assert np.array_equal(e2, eta) and np.array_equal(c2, chi)
    wz = copy.copy(wl)
    wz.vel = np.zeros_like(wl.vel)
    ea, _ = orc.direction_fields(wz, wl.dirs[0])
    eb, _ = orc.direction_fields(wz, wl.dirs[4])
    assert np.array_equal(ea, eb)
    assert not np.array_equal(orc.direction_fields(wl, wl.dirs[0])[0], orc.direction_fields(wl, wl.dirs[4])[0])
    # (iii)
    A = orc.plain_march(wl, variant=orc.CLASSIC)
    JA = orc.mean_intensity(A.I, wl.weights)
    w0 = copy.copy(wl)
    w0.max_level = 0
    J0, lv0, seg0 = orc.single_direction_solve(w0)
    assert (lv0[:, :, act] == 0).all() and (lv0[:, :, ~act] == -1).all()
    assert seg0 == orc.hdda_march(wl, orc.build_mips(wl, max_level=0)).segments      # same non-empty visits
    assert max_rel(J0, JA) < 3e-7
    # (iv)
    wv = copy.copy(wl)
    wv.thr_eta = wv.thr_chi = 0.3
    J1, lv1, seg1 = orc.single_direction_solve(wv)
    assert lv1.shape == (wl.dirs.shape[0], wl.n_batch, act.shape[0])
    assert (lv1 > 0).any() and seg1 < seg0
    assert any(not np.array_equal(lv1[0], lv1[k]) for k in range(1, lv1.shape[0]))
    s3 = orc.single_direction_workload(wv, 3)
    assert np.array_equal(orc.build_mips(s3, variant=orc.ISO).levels, lv1[3])
    assert np.percentile(np.abs(J1 - JA) / JA, 99) < 0.2


# ------------------------------------------------------------------------------------------------
# P14-P17: the anisotropic VLM tests and the velocity-table pyramid (V6, R-vel).  Every C3 / C4 / C5
# level table -- hence every timed segment count -- hangs on these three readings.
# ------------------------------------------------------------------------------------------------
def _one_line_medium(n, u_kms, vth_kms, speeds_x, chi_star=None, n_vbins=9, max_level=1, thr=1e-2):
    """Hand-controlled one-line moving medium on an n x n grid (brick 16, all active): uniform line parameters
    (a = 0.01, thermal width vth_kms), wavelengths at Doppler offsets u_kms from the line centre, velocity (speeds_x, 0)
    per voxel, no background.  Everything of C3's generated fields is overwritten."""
    wl = make("C3", n=n, n_dirs=4, n_probes=4, n_lambda=len(u_kms), max_level=max_level, n_vbins=n_vbins)
    nv = n * n
    lam0 = 500.0
    wl.active[:] = 1
    wl.lam = (lam0 * (1.0 + np.asarray(u_kms, dtype=np.float64) / wl.c_light)).astype(np.float32)
    wl.lambda0 = np.array([lam0], dtype=np.float32)
    dlamD = lam0 * vth_kms / wl.c_light
    cs = np.full(nv, 2.0) if chi_star is None else np.asarray(chi_star, dtype=np.float64).ravel()
    wl.chi_star0 = (cs * math.sqrt(math.pi) * dlamD).astype(np.float32)[None, :]
    wl.eta_star0 = (1.5 * wl.chi_star0).astype(np.float32)
    wl.a0 = np.full((1, nv), 0.01, dtype=np.float32)
    wl.inv_dlamD = np.full((1, nv), 1.0 / dlamD, dtype=np.float32)
    wl.eta_bg = np.zeros((nv, len(u_kms)), dtype=np.float32)
    wl.chi_bg = np.zeros((nv, len(u_kms)), dtype=np.float32)
    wl.vel = np.zeros((nv, 2), dtype=np.float32)
    wl.vel[:, 0] = np.asarray(speeds_x, dtype=np.float32).ravel()
    wl.thr_eta = wl.thr_chi = thr
    return wl


def test_p14_cav_test_quantity_is_the_worst_case_shift_brute_force():
    """eq. 17: the Core-and-Voigt VLM test sums, per line, the terms "Doppler shifted to the
    wavelength closest to the line core possible in the current voxel".  Brute force, independent of the oracle's
    clamp formula: (i) over 401 velocities in [-V, V], |lam0 (1 - v/c) - lam| is never smaller than at the oracle's
    v_D; (ii) the test quantity of build_mips (cav_test_fields) equals background + sum over the active lines of the
    MAXIMUM over those velocities of the textbook line term (scipy's Faddeeva function, not HUM1WEI24): the line
    opacity falls monotonically away from the core, so the closest shift is the strongest one."""
    from scipy.special import wofz
    wl = make("C4", n=64, n_dirs=4, n_probes=4)
    M = orc.build_mips(wl, max_level=2)
    c = wl.c_light
    rng = np.random.default_rng(17)
    n_clamped = n_free = n_pos = n_neg = 0
    for m in (0, 1, 2):
        te, tc = orc.cav_test_fields(wl, M, m)
        shape = orc.grid_shape(wl, m)
        V = M.vmax[m].astype(np.float64)
        cells = np.argwhere(M.chi_star[m][0] > 0)
        pick = cells[rng.choice(len(cells), size=min(60, len(cells)), replace=False)]
        for (cy, cx) in pick:
            Vc = float(V[cy, cx])
            vgrid = np.linspace(-Vc, Vc, 401)
            for j in rng.choice(wl.n_lambda, size=24, replace=False):
                b = j // wl.lambda_batch
                lam = float(wl.lam[j])
                e_max, c_max = float(M.eta[m][cy, cx, j]), float(M.chi[m][cy, cx, j])
                lines = [int(q) for q in wl.active_lines[b] if q >= 0]
                for l in lines:
                    lam0 = float(wl.lambda0[l])
                    vD = float(orc.cav_worst_case_shift(np.array([lam]), lam0, np.array([Vc]), c)[0, 0])
                    assert -Vc <= vD <= Vc
                    f = np.abs(lam0 * (1.0 - vgrid / c) - lam)
                    assert abs(lam0 * (1.0 - vD / c) - lam) <= f.min() * (1 + 1e-12) + 1e-12
                    n_clamped += abs(vD) == Vc
                    n_free += abs(vD) < Vc
                    n_pos += vD > 0
                    n_neg += vD < 0
                    inv = float(M.inv_dlamD[m][l][cy, cx])
                    x = (lam - lam0 + vgrid / c * lam0) * inv
                    a = (lam / lam0) ** 2 * float(M.a0[m][l][cy, cx])
                    phi = wofz(x + 1j * a).real * inv / math.sqrt(math.pi)
                    e_max += lam0 / lam * float(M.eta_star[m][l][cy, cx]) * phi.max()
                    c_max += lam0 / lam * float(M.chi_star[m][l][cy, cx]) * phi.max()
                # the grid maximum can only fall short of the true one by the grid spacing: (dx/2)^2 with dx the step
                # in Doppler widths; HUM1WEI24 against wofz: 3e-6 in the far wings (P13)
                dx = max([(2.0 * Vc / 400.0) / c * float(wl.lambda0[l]) * float(M.inv_dlamD[m][l][cy, cx]) for l in lines] + [0.0])
                slack = 3e-6 + 0.3 * dx * dx
                assert c_max * (1 - 3e-6) <= tc[cy, cx, j] <= c_max * (1 + slack), (m, cy, cx, j)
                assert e_max * (1 - 3e-6) <= te[cy, cx, j] <= e_max * (1 + slack), (m, cy, cx, j)
    assert min(n_clamped, n_free, n_pos, n_neg) > 50        # both regimes and both signs were exercised


def test_p14_cav_level_decision_hand_example():
    """eq. 17 on a hand example: one line, thermal width 10 km/s, eight wavelengths 0.25 .. 2 km/s redward of the
    core; columns alternate |v| = 1 and 2 km/s, so every level-1 cell has children (1, 2, 1, 2) km/s.  Shifted TOWARDS
    the core the reddest wavelength sits at x = (2 - 1)/10 = 0.1 in the slow children and at x = 0 in the fast ones:
    H = e^-0.01 against 1, relative variance (0.005 / 0.995)^2 = 2.5e-5.  (Shifted AWAY from the core it would be
    x = 0.3 against 0.4: 1.2e-3.)  So the brick coarsens at a threshold of 2e-4 and does not at 1e-5."""
    n = 16
    u = 0.25 * np.arange(1, 9)
    speeds = np.where(np.arange(n)[None, :] % 2 == 0, 1.0, 2.0) * np.ones((n, 1))
    wl = _one_line_medium(n, u, 10.0, speeds)
    assert (orc.build_mips(wl, variant=orc.CAV, thr_eta=2e-4, thr_chi=2e-4).levels == 1).all()
    assert (orc.build_mips(wl, variant=orc.CAV, thr_eta=1e-5, thr_chi=1e-5).levels == 0).all()
    # the same blueward of the core (the other sign of v_D)
    wl = _one_line_medium(n, -u, 10.0, speeds)
    assert (orc.build_mips(wl, variant=orc.CAV, thr_eta=2e-4, thr_chi=2e-4).levels == 1).all()
    assert (orc.build_mips(wl, variant=orc.CAV, thr_eta=1e-5, thr_chi=1e-5).levels == 0).all()
    # every wavelength within reach of every child's velocity range: all children are tested AT the core, where a
    # medium with uniform line parameters is uniform -- coarsens at any positive threshold
    wl = _one_line_medium(n, u, 10.0, speeds * 3.0)
    assert (orc.build_mips(wl, variant=orc.CAV, thr_eta=1e-9, thr_chi=1e-9).levels == 1).all()


def test_p15_max_speed_chain_hand_example():
    """PAPER.md:196 / :311: the velocity range of a MIP N voxel is taken "over the set of voxels MIP 0 contained
    within" it: max |v| of the children, level by level.  4 x 4 typed-in speeds (3-4-5 triangles)."""
    a = np.array([[1, 5, 2, 2], [3, 4, 2, 9], [7, 1, 1, 1], [0, 6, 1, 8]], dtype=np.float32)
    assert np.array_equal(orc.mip_max(a, 2), np.array([[5, 9], [7, 8]], dtype=np.float32))
    assert np.array_equal(orc.mip_max(orc.mip_max(a, 2), 2), np.array([[9]], dtype=np.float32))
    a3 = np.zeros((2, 2, 2), dtype=np.float32)
    a3[1, 0, 1] = 4.0
    a3[0, 1, 0] = 2.5
    assert np.array_equal(orc.mip_max(a3, 3), np.array([[[4.0]]], dtype=np.float32))
    # through build_mips: speeds are the Euclidean norm of the velocity, (3, 4) -> 5
    n = 16
    wl = _one_line_medium(n, np.linspace(-20, 20, 8), 10.0, np.zeros((n, n)), max_level=2)
    vx = np.zeros((n, n))
    vy = np.zeros((n, n))
    vx[5, 6], vy[5, 6] = 3.0, -4.0
    vx[0, 0] = -2.0
    wl.vel[:, 0], wl.vel[:, 1] = vx.ravel(), vy.ravel()
    M = orc.build_mips(wl, variant=orc.CAV)
    assert M.vmax[0][5, 6] == 5.0 and M.vmax[1][2, 3] == 5.0 and M.vmax[2][1, 1] == 5.0
    assert M.vmax[1][0, 0] == 2.0 and M.vmax[2][0, 0] == 2.0
    assert M.vmax[1].sum() == 7.0 and M.vmax[2].sum() == 7.0          # and nothing anywhere else
    # the box-filtered velocity (what the ray projects) is the mean, not the max
    assert M.vbar[1][2, 3, 0] == 0.75 and M.vbar[1][2, 3, 1] == -1.0 and M.vbar[2][1, 1, 0] == 0.1875


def test_p16_velocity_table_pyramid():
    """R-vel (the higher levels are not spelled out).  (i) Hand example: five bins, children
    A (V = 10, nodes -10 -5 0 5 10) and B (V = 20, nodes -20 .. 20), twice each; the parent spans [-20, 20] and each
    child is read ON ITS OWN grid, clamped: at v = -10 child A gives its first node, not its second.  (ii) Children
    with equal V and equal tables reproduce themselves bit for bit.  (iii) On a generated atmosphere every parent
    table equals the mean of numpy.interp over explicit child grids (a library routine, clamping at the ends).
    (iv) A static medium (v = 0) with mips on: level tables and intensities of the velocity-interpolation build equal
    those of the ISO build of the rest-frame fields."""
    A = np.array([1.0, 2.0, 4.0, 8.0, 16.0], dtype=np.float32)
    B = np.array([32.0, 64.0, 128.0, 256.0, 512.0], dtype=np.float32)

    def tab(vals):                       # one cell, 5 bins, 1 wavelength, (eta, chi) = (vals, 3 vals)
        return np.stack([vals, 3 * vals], axis=-1).reshape(1, 5, 1, 2).astype(np.float32)

    V = lambda v: np.array([v], dtype=np.float32)
    parent = orc.velinterp_parent_table([tab(A), tab(B), tab(A), tab(B)], [V(10), V(20), V(10), V(20)], V(20), 5)
    # parent bins -20 -10 0 10 20: A -> 1 1 4 16 16 (clamped outside its +-10), B -> its own nodes
    want = (np.array([1, 1, 4, 16, 16]) + np.array([32, 64, 128, 256, 512])) / 2.0
    assert np.array_equal(parent[0, :, 0, 0], want.astype(np.float32))
    assert np.array_equal(parent[0, :, 0, 1], (3 * want).astype(np.float32))
    # between nodes: child A (V = 10) at parent bins of V = 16: -16 -8 0 8 16 -> 1, 1.4, 4, 12.8, 16
    parent = orc.velinterp_parent_table([tab(A)] * 4, [V(10)] * 4, V(16), 5)
    assert np.allclose(parent[0, :, 0, 0], [1.0, 1.4, 4.0, 12.8, 16.0], rtol=1e-7)
    # (ii)
    same = orc.velinterp_parent_table([tab(B)] * 4, [V(20)] * 4, V(20), 5)
    assert np.array_equal(same, tab(B))
    wl = make("C3", n=64, n_dirs=4, n_probes=30, max_level=3)
    for name in ("eta_bg", "chi_bg", "vel"):
        a = getattr(wl, name).reshape(64, 64, -1)
        setattr(wl, name, np.ascontiguousarray(np.repeat(np.repeat(a[::2, ::2], 2, axis=0), 2, axis=1).reshape(64 * 64, -1)))
    for name in ("eta_star0", "chi_star0", "a0", "inv_dlamD"):
        a = getattr(wl, name).reshape(1, 64, 64)
        setattr(wl, name, np.ascontiguousarray(np.repeat(np.repeat(a[:, ::2, ::2], 2, axis=1), 2, axis=2).reshape(1, -1)))
    M2 = orc.build_mips(wl)
    assert np.array_equal(M2.vtab[1], M2.vtab[0][::2, ::2]) and np.array_equal(M2.vmax[1], M2.vmax[0][::2, ::2])
    # (iii)
    wl = make("C3", n=64, n_dirs=4, n_probes=30, max_level=3)
    M = orc.build_mips(wl)
    nb = wl.n_vbins
    rng = np.random.default_rng(23)
    differs = 0
    for m in (1, 2, 3):
        ny, nx = orc.grid_shape(wl, m)
        for _ in range(40):
            cy, cx = int(rng.integers(ny)), int(rng.integers(nx))
            Vp = float(M.vmax[m][cy, cx])
            if Vp == 0.0:
                continue
            vk = np.linspace(-Vp, Vp, nb)
            kids = [(2 * cy + dy, 2 * cx + dx) for dy in (0, 1) for dx in (0, 1)]
            assert Vp == max(float(M.vmax[m - 1][k]) for k in kids)
            for j in rng.choice(wl.n_lambda, size=5, replace=False):
                for q in (0, 1):
                    acc = np.zeros(nb)
                    for k in kids:
                        Vc = float(M.vmax[m - 1][k])
                        vals = M.vtab[m - 1][k][:, j, q].astype(np.float64)
                        acc += np.interp(vk, np.linspace(-Vc, Vc, nb), vals) if Vc > 0 else vals[0]
                        differs += Vc < 0.9 * Vp
                    assert np.allclose(M.vtab[m][cy, cx, :, j, q], acc / 4.0, rtol=3e-7, atol=0)
    assert differs > 100                                      # children whose range is well inside the parent's
    # (iv)
    ws = make("C3", n=64, n_dirs=6, n_probes=40, max_level=3)
    ws.vel[:] = 0.0
    ws.thr_eta = ws.thr_chi = 0.2                               # a mix of levels 1 and 2 on this 64^2 atmosphere
    Mv = orc.build_mips(ws)
    assert Mv.levels.max() >= 2 and (Mv.levels == 1).any()
    rest = Mv.vtab[0][:, :, 0]                                  # [ny][nx][lambda][2]: every bin holds the static value
    assert all(np.array_equal(Mv.vtab[0][:, :, k], rest) for k in range(ws.n_vbins))
    iso = iso_workload((64, 64), ws.brick, rest[..., 0], rest[..., 1], ws.probe_pos, ws.dirs, active=ws.active,
                       max_level=3, thr=0.2)
    Mi = orc.build_mips(iso)
    assert np.array_equal(Mi.levels, Mv.levels)
    a, b = orc.hdda_march(ws, Mv, capture_batch=0), orc.hdda_march(iso, Mi, capture_batch=0)
    assert np.array_equal(a.records, b.records) and max_rel(a.I, b.I) < 1e-14


def test_p17_velinterp_tests_the_rest_frame():
    """the level test of the velocity-interpolation scheme is "computed ... using the values ... in the
    rest frame of each voxel (i.e. the centre of the velocity grid, with a velocity of 0)".  A medium whose line
    parameters are uniform but whose speeds differ from voxel to voxel is uniform at rest and varies in every shifted
    bin: it must coarsen fully.  The converse -- uniform speeds, line strength varying 1 : 3 inside every level-1
    cell -- must not coarsen.  (Nine bins: the centre node is v = 0 exactly.)"""
    n = 16
    u = np.linspace(-20.0, 20.0, 8)
    rng = np.random.default_rng(4)
    speeds = rng.uniform(2.0, 25.0, size=(n, n))
    wl = _one_line_medium(n, u, 10.0, speeds, n_vbins=9, max_level=4)
    M = orc.build_mips(wl, variant=orc.VELINTERP)
    assert (M.levels == 4).all()
    last = M.vtab[0][:, :, -1, :, 1]                           # the shifted bins do vary (by far more than 1e-2)
    assert (last.std(axis=(0, 1)) / last.mean(axis=(0, 1))).max() > 0.1
    e0, c0 = orc.velinterp_rest_frame(M.vtab[0], M.vmax[0], 9)
    assert (c0 == c0[0, 0]).all() and (e0 == e0[0, 0]).all()
    cs = np.where(np.arange(n)[:, None] % 2 == 0, 1.0, 3.0) * np.ones((1, n))
    wl = _one_line_medium(n, u, 10.0, np.full((n, n), 7.0), chi_star=cs, n_vbins=9, max_level=4, thr=0.2)
    assert (orc.build_mips(wl, variant=orc.VELINTERP).levels == 0).all()        # relvar of (1,1,3,3) is 0.25 > 0.2
    wl.thr_eta = wl.thr_chi = 0.26
    assert (orc.build_mips(wl, variant=orc.VELINTERP).levels >= 1).all()


# ------------------------------------------------------------------------------------------------
# The 3D half of the level selection (SURVEY.md 8(c) V1, V2, V5, P7, P10; PAPER.md:127-130 eq. 8, :142, :148).
# Mutants these pins exist for: sample instead of population variance over the 8 children,
# and a brick aggregation with two brick axes exchanged.
# ------------------------------------------------------------------------------------------------
def _iso_3d_from_c5(n=32, n_dirs=6, n_probes=40, seed=5):
    """C5's occupancy, probes and directions around a static (ISO) 3D medium: a smooth stratification times log-normal
    small-scale noise whose amplitude is drawn per brick (0 / 1 % / 5 % / 30 %) and grows with wavelength, so that
    bricks and wavelength batches land on different levels.  Input recipe only: no method arithmetic."""
    wl = make("C5", n=n, n_dirs=n_dirs, n_probes=n_probes)
    rng = np.random.default_rng(seed)
    b = wl.brick
    nb = n // b
    z = np.arange(n, dtype=np.float64)[:, None, None, None]
    base = np.exp(-np.abs(z - n / 2.0) / (2.0 * n)) * np.ones((n, n, n, 1))
    amp_b = rng.choice([0.0, 0.01, 0.05, 0.3], size=(nb, nb, nb))
    amp = np.repeat(np.repeat(np.repeat(amp_b, b, 0), b, 1), b, 2)[..., None] * np.linspace(0.25, 1.0, wl.n_lambda)
    occ = wl.active.reshape(n, n, n, 1).astype(bool)
    eta = base * np.exp(amp * rng.standard_normal((n, n, n, wl.n_lambda))) * occ
    chi = 0.3 * base * np.exp(amp * rng.standard_normal((n, n, n, wl.n_lambda))) * occ
    return iso_workload((n, n, n), b, eta, chi, wl.probe_pos, wl.dirs, active=wl.active, weights=wl.weights,
                        max_level=3, h=wl.voxel_size)


def _levels_by_loops_3d(wl, max_level, metric, thr, tau_gate):
    """Second implementation of V1-V5 for a 3D ISO medium, structured brick by brick: each populated brick builds its
    own little pyramid in python floats and stops at the first level where one of its cells fails.  The statistic is
    typed out for 8 children with the population variance (divide by 8, eq. 8 / V2), the mean as the V1 child-order sum
    times 1/8 rounded once to fp32."""
    nx, ny, nz = wl.dims
    B, W, h = wl.brick, wl.lambda_batch, float(wl.voxel_size)
    thr, tau_gate = float(np.float32(thr)), float(np.float32(tau_gate))
    eta = wl.eta.reshape(nz, ny, nx, wl.n_lambda)
    chi = wl.chi.reshape(nz, ny, nx, wl.n_lambda)
    act = wl.active.reshape(nz, ny, nx)
    nbx, nby, nbz = nx // B, ny // B, nz // B
    out = np.zeros((wl.n_batch, nbx * nby * nbz), dtype=np.int8)

    def kids(p, k, j, i, l):      # child order: x fastest, then y, then z (V1)
        return [float(p[2 * k + dz, 2 * j + dy, 2 * i + dx, l]) for dz in (0, 1) for dy in (0, 1) for dx in (0, 1)]

    def total(v):
        return ((((((v[0] + v[1]) + v[2]) + v[3]) + v[4]) + v[5]) + v[6]) + v[7]

    def stat(vals):
        if all(v == vals[0] for v in vals):
            return 0.0
        if metric == orc.IOD_LOG:
            if any(v <= 0 for v in vals):
                return math.inf
            X = [math.log(v * h) for v in vals]
        else:
            X = list(vals)
        mean = total(X) / 8
        var = total([(x - mean) ** 2 for x in X]) / 8            # population variance of the 8 children
        if mean == 0:
            return math.inf
        return abs(var / mean) if metric == orc.IOD_LOG else var / (mean * mean)

    for bz in range(nbz):
        for by in range(nby):
            for bx in range(nbx):
                bi = (bz * nby + by) * nbx + bx
                box = (slice(bz * B, (bz + 1) * B), slice(by * B, (by + 1) * B), slice(bx * B, (bx + 1) * B))
                if not act[box].any():
                    out[:, bi] = -1
                    continue
                for bt in range(wl.n_batch):
                    pe = eta[box][..., bt * W:(bt + 1) * W].astype(np.float64)
                    pc = chi[box][..., bt * W:(bt + 1) * W].astype(np.float64)
                    level = 0
                    for m in range(1, max_level + 1):
                        s = pe.shape[0] // 2
                        ne, nc = np.zeros((s, s, s, W)), np.zeros((s, s, s, W))
                        ok = True
                        for k in range(s):
                            for j in range(s):
                                for i in range(s):
                                    for l in range(W):
                                        ve, vc = kids(pe, k, j, i, l), kids(pc, k, j, i, l)
                                        ne[k, j, i, l] = np.float32(total(ve) * 0.125)
                                        nc[k, j, i, l] = np.float32(total(vc) * 0.125)
                                        passed = stat(ve) < thr and stat(vc) < thr
                                        if tau_gate >= 0 and (total(vc) / 8) * h <= tau_gate:
                                            passed = True
                                        ok = ok and passed
                        if not ok:
                            break
                        level, pe, pc = m, ne, nc
                    out[bt, bi] = level
    return out


@pytest.mark.parametrize("metric,thr,gate", [(orc.RELVAR, 1e-3, -1.0), (orc.RELVAR, 1e-4, -1.0),
                                             (orc.IOD_LOG, 0.02, 0.2), (orc.IOD_LOG, 0.004, -1.0)])
def test_p10_3d_level_selection_second_implementation(metric, thr, gate):
    wl = _iso_3d_from_c5()
    M = orc.build_mips(wl, max_level=3, metric=metric, thr_eta=thr, thr_chi=thr, tau_gate=gate)
    ref = _levels_by_loops_3d(wl, 3, metric, thr, gate)
    assert (ref == -1).any() and len(np.unique(ref[ref >= 0])) >= 2      # the case separates levels
    assert np.array_equal(M.levels, ref)


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_p10_3d_hand_example_population_variance(axis):
    """2x2x2 children (1,1,1,1,3,3,3,3), the 3s on the upper half along `axis` (numpy order z, y, x): mean 2, population
    variance 1 -> relvar 1/4 (the sample variance 8/7 would give 2/7 = 0.2857); X = ln x = (0 x4, ln3 x4): mean ln3/2,
    variance (ln3/2)^2 -> IoD = ln3/2 = 0.5493 (sample variance: 0.6278)."""
    dims = (8, 8, 8)
    x = np.ones(dims)
    sl = [slice(None)] * 3
    sl[axis] = slice(1, None, 2)
    x[tuple(sl)] = 3.0
    wl = iso_workload(dims, 8, x, x, [[1.5, 1.5, 1.5]], [[1.0, 0.0, 0.0]], max_level=3)
    assert (orc.build_mips(wl, metric=orc.RELVAR, thr_eta=0.2501, thr_chi=0.2501).levels >= 1).all()
    assert (orc.build_mips(wl, metric=orc.RELVAR, thr_eta=0.2499, thr_chi=0.2499).levels == 0).all()
    assert (orc.build_mips(wl, metric=orc.IOD_LOG, thr_eta=0.5494, thr_chi=0.5494).levels >= 1).all()
    assert (orc.build_mips(wl, metric=orc.IOD_LOG, thr_eta=0.5492, thr_chi=0.5492).levels == 0).all()
    # level-1 cells are all 2 -> once level 1 passes every higher level does (IoD = 0 < thr)
    assert (orc.build_mips(wl, metric=orc.RELVAR, thr_eta=0.2501, thr_chi=0.2501).levels == 3).all()
    # the statistic itself, on one cell: children in V1 order
    ch = [np.array([v], dtype=np.float64) for v in (1, 1, 1, 1, 3, 3, 3, 3)]
    assert orc.cell_metric(ch, orc.RELVAR, 1.0)[0] == 0.25
    assert abs(orc.cell_metric(ch, orc.IOD_LOG, 1.0)[0] - math.log(3.0) / 2) < 1e-15
    # gate: mean chi h = 2
    assert (orc.build_mips(wl, metric=orc.RELVAR, thr_eta=0.0, thr_chi=0.0, tau_gate=2.0).levels == 3).all()
    assert (orc.build_mips(wl, metric=orc.RELVAR, thr_eta=0.0, thr_chi=0.0, tau_gate=1.99).levels == 0).all()


def test_p10_3d_brick_aggregation_typed_in_levels():
    """A 4 x 3 x 2 brick lattice (x, y, z) whose bricks are told apart by position: brick b = (bz*3 + by)*4 + bx (V5,
    PAPER.md:148, :170).  Smooth everywhere (level 3) except four marked bricks; exchanging any two brick axes in the
    aggregation moves the marks (or cannot even be reshaped)."""
    nx, ny, nz, B = 32, 24, 16, 8
    x = np.full((nz, ny, nx), 0.5)
    act = np.ones((nz, ny, nx), dtype=np.uint8)

    def box(bx, by, bz):
        return (slice(bz * B, (bz + 1) * B), slice(by * B, (by + 1) * B), slice(bx * B, (bx + 1) * B))

    # (3, 1, 0): one odd voxel -> its level-1 cell fails -> level 0
    v = x[box(3, 1, 0)]; v[5, 2, 7] = 5.0
    # (0, 2, 1): constant 2^3 blocks, one block different -> level 1 passes, its level-2 cell fails -> level 1
    v = x[box(0, 2, 1)]; v[2:4, 6:8, 0:2] = 5.0
    # (2, 0, 1): constant 4^3 blocks, one different -> levels 1, 2 pass, level 3 fails -> level 2
    v = x[box(2, 0, 1)]; v[4:8, 0:4, 4:8] = 5.0
    # (1, 2, 0): no active voxel -> empty
    act[box(1, 2, 0)] = 0
    want = np.full(4 * 3 * 2, 3, dtype=np.int8)
    want[(0 * 3 + 1) * 4 + 3] = 0      # brick 7
    want[(1 * 3 + 2) * 4 + 0] = 1      # brick 20
    want[(1 * 3 + 0) * 4 + 2] = 2      # brick 14
    want[(0 * 3 + 2) * 4 + 1] = -1     # brick 9
    wl = iso_workload((nx, ny, nz), B, x, x, [[1.5, 1.5, 1.5]], [[1.0, 0.0, 0.0]], active=act.ravel(), max_level=3)
    for metric in (orc.RELVAR, orc.IOD_LOG):
        M = orc.build_mips(wl, max_level=3, metric=metric, thr_eta=1e-3, thr_chi=1e-3)
        assert M.levels.shape == (1, 24)
        assert np.array_equal(M.levels[0], want)
    # occupancy in the same numbering
    assert np.array_equal(orc.brick_active(wl), want >= 0)


def test_v1_3d_mip_values_are_correctly_rounded_means():
    rng = np.random.default_rng(4)
    a = np.exp(rng.standard_normal((4, 6, 8, 2)) * 4).astype(np.float32)       # (z, y, x, channel), all sides differ
    m = orc.mip_mean(a, 3)
    assert m.shape == (2, 3, 4, 2)
    from fractions import Fraction
    for k in range(2):
        for j in range(3):
            for i in range(4):
                for c in range(2):
                    ex = sum(Fraction(float(a[2 * k + dz, 2 * j + dy, 2 * i + dx, c]))
                             for dz in (0, 1) for dy in (0, 1) for dx in (0, 1)) / 8
                    assert float(m[k, j, i, c]) == float(np.float32(float(ex)))


def test_p7_3d_hdda_equals_plain_march_over_upsampled_field():
    """P7 in 3D: segments of equal eta, chi compose exactly, so the VLM + HDDA solve equals the plain level-0 march
    through the field in which every voxel carries the mip value of the cell its brick's level puts it in."""
    wl = _iso_3d_from_c5(n=32, n_dirs=8, n_probes=60)
    M = orc.build_mips(wl, max_level=3, metric=orc.RELVAR, thr_eta=1e-3, thr_chi=1e-3)
    assert len(np.unique(M.levels[M.levels >= 0])) >= 3
    Bm = orc.hdda_march(wl, M)
    n, b, W = 32, wl.brick, wl.lambda_batch
    eta_up = np.zeros((n, n, n, wl.n_lambda), dtype=np.float32)
    chi_up = np.zeros_like(eta_up)
    nbk = n // b
    for bt in range(wl.n_batch):
        sl = slice(bt * W, (bt + 1) * W)
        for bi in range(wl.n_bricks):
            m = int(M.levels[bt, bi])
            if m < 0:
                continue
            bz, r = divmod(bi, nbk * nbk)
            by, bx = divmod(r, nbk)
            cb = b >> m
            for name, up in (("eta", eta_up), ("chi", chi_up)):
                src = getattr(M, name)[m][bz * cb:(bz + 1) * cb, by * cb:(by + 1) * cb, bx * cb:(bx + 1) * cb, sl]
                for ax in range(3):
                    src = np.repeat(src, 1 << m, axis=ax)
                up[bz * b:(bz + 1) * b, by * b:(by + 1) * b, bx * b:(bx + 1) * b, sl] = src
    wl_up = iso_workload((n, n, n), b, eta_up, chi_up, wl.probe_pos, wl.dirs, active=wl.active, weights=wl.weights)
    A = orc.plain_march(wl_up)
    assert Bm.segments < A.segments
    assert max_rel(Bm.I, A.I) < 2e-6
