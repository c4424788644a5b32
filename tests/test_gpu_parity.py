"""GPU parity: the CUDA path behind the C ABI against the CPU oracle on the same seeded inputs.

Bars (BASELINE.json north_star): level tables and mip values bit-exact, traversal index lists (and
their fp32 path lengths) bit-exact, intensities and J within 1e-5 max relative error in fp32.
"""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import oracle as orc           # noqa: E402
from workloads import make                 # noqa: E402
from workloads.gen import dirs_2d          # noqa: E402
from _util import (batch_workload, crop_brick_ids, crop_workload, fig5_levels, iso_workload, max_rel, random_unit_dirs,   # noqa: E402
                   unit_dirs_2d)

TOL = 1e-5


@pytest.fixture(scope="module")
def P():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2511_08498_b200 as pkg
    # the tests run the production mapping (one thread per ray) unless they say otherwise; the library's default is
    # automatic (8 lanes per ray for problems smaller than one wave of blocks), exercised by test_c1_full
    pkg.dex_set_lanes_per_ray(1)
    return pkg


def _build(P, wl, **ov):
    dw = P.pipeline.upload(wl, "cuda:0")
    grid = P.pipeline.build_grid(dw)
    mips = P.pipeline.build_mips(dw, grid, **ov)
    return dw, grid, mips


def _check_build(P, wl, M, grid, mips, spectra=True):
    act = orc.brick_active(wl)
    slots = grid.slots()
    assert np.array_equal(slots >= 0, act)
    assert np.array_equal(np.sort(slots[slots >= 0]), np.arange(int(act.sum())))
    lv = mips.levels()
    assert np.array_equal(lv, M.levels), f"level tables differ in {(lv != M.levels).sum()} entries"
    if spectra:
        for m in range(M.max_level + 1):
            for chain, ref in ((P.DEX_CHAIN_ETA, M.eta[m]), (P.DEX_CHAIN_CHI, M.chi[m])):
                got = mips.level_data(chain, m)
                mask = _active_cell_mask(wl, act, m)
                assert np.array_equal(got[mask].view(np.uint32), np.ascontiguousarray(ref)[mask].view(np.uint32))
    for b in range(wl.n_batch):
        assert np.array_equal(mips.packed_levels(b), orc.pack_levels(M.levels[b], M.max_level))


def _active_cell_mask(wl, act_b, m):
    cb = wl.brick >> m
    bd = wl.brick_dims
    if wl.ndim == 2:
        a = act_b.reshape(bd[1], bd[0])
        return np.repeat(np.repeat(a, cb, axis=0), cb, axis=1)
    a = act_b.reshape(bd[2], bd[1], bd[0])
    return np.repeat(np.repeat(np.repeat(a, cb, axis=0), cb, axis=1), cb, axis=2)


def _check_lists(cap, res, room):
    counts = cap.counts.cpu().numpy()
    assert np.array_equal(counts, res.counts)
    rec = cap.records.cpu().numpy().view(np.uint64).reshape(-1, room)
    ds = cap.ds.cpu().numpy().reshape(-1, room)
    for r in range(counts.shape[0]):
        n = counts[r]
        assert np.array_equal(rec[r, :n], res.records[r, :n]), f"ray {r}: records differ"
        assert np.array_equal(ds[r, :n].view(np.uint32), res.ds[r, :n].view(np.uint32)), f"ray {r}: ds differ"


def _solve_and_compare(P, wl, M, dw, grid, mips, capture_batches=(0,), lanes=(8, 4, 2, 1), tol=TOL):
    ref = None
    for cb in capture_batches:
        res = orc.hdda_march(wl, M, capture_batch=cb)
        ref = res
        I, cap = P.pipeline.formal_solution(dw, grid, mips, capture_batch=cb, want_I=False)
        _check_lists(cap, res, cap.room)
    Jref = orc.mean_intensity(ref.I, wl.weights)
    for lpr in lanes:
        P.dex_set_lanes_per_ray(lpr)
        seg = torch.zeros(1, dtype=torch.int64, device="cuda:0")
        I, _ = P.pipeline.formal_solution(dw, grid, mips, segment_count=seg)
        assert int(seg.item()) == ref.segments
        assert max_rel(I.cpu().numpy(), ref.I) <= tol, f"lanes={lpr}"
        seg.zero_()
        J = P.pipeline.mean_intensity(dw, grid, mips, segment_count=seg)
        assert int(seg.item()) == ref.segments
        assert max_rel(J.cpu().numpy(), Jref) <= tol
        J2 = torch.empty_like(J)
        P.dex_mean_intensity(grid, mips, P.pipeline.rays(dw), J2, I)
        assert max_rel(J2.cpu().numpy(), Jref) <= tol
    P.dex_set_lanes_per_ray(1)
    return ref


# ------------------------------------------------------------------------------------------ ISO
def test_c1_full(P):
    """configs[0]: 64x64 dense, 8 wavelengths, 16 directions, a probe at every voxel centre."""
    wl = make("C1")
    M = orc.build_mips(wl)
    dw, grid, mips = _build(P, wl)
    _check_build(P, wl, M, grid, mips)
    ref = _solve_and_compare(P, wl, M, dw, grid, mips)
    P.dex_set_lanes_per_ray(0)             # automatic: 4096 probes < one wave of blocks -> 8 lanes per ray
    try:
        J = P.pipeline.mean_intensity(dw, grid, mips)
        assert max_rel(J.cpu().numpy(), orc.mean_intensity(ref.I, wl.weights)) <= TOL
    finally:
        P.dex_set_lanes_per_ray(1)


@pytest.mark.parametrize("metric,thr,gate", [(1, 1e-2, -1.0), (0, 1.0, 0.25), (1, 0.0, -1.0)])
def test_c2_small_with_mips(P, metric, thr, gate):
    wl = make("C2", n=256, n_dirs=16, n_probes=1500)
    d0, _ = dirs_2d(8, phase=0.0)           # axis-aligned and exact diagonals
    wl.dirs = np.concatenate([wl.dirs, d0]).astype(np.float32)
    wl.weights = np.full(len(wl.dirs), 1.0 / len(wl.dirs), dtype=np.float32)
    wl.metric, wl.thr_eta, wl.thr_chi, wl.tau_gate = metric, thr, thr, gate
    M = orc.build_mips(wl)
    dw, grid, mips = _build(P, wl)
    _check_build(P, wl, M, grid, mips)
    _solve_and_compare(P, wl, M, dw, grid, mips, capture_batches=(0, 1))


def test_iso_3d_with_mips(P):
    wl = make("C5", n=64, n_dirs=12, n_probes=600)
    wl.variant = 0
    wl.eta, wl.chi = wl.eta_bg, wl.chi_bg
    wl.thr_eta = wl.thr_chi = 1.0
    M = orc.build_mips(wl)
    assert M.levels.max() >= 2
    dw, grid, mips = _build(P, wl)
    _check_build(P, wl, M, grid, mips)
    _solve_and_compare(P, wl, M, dw, grid, mips)


def test_fig5_fixture_injected_levels_and_boundary_intensity(P):
    """Fig. 5 block states injected through dex_mips_set_levels; nonzero incoming intensity."""
    rng = np.random.default_rng(8)
    lv = fig5_levels()
    probes = np.concatenate([rng.uniform(0, 32, size=(40, 2)), [[16.5, 16.5], [0.5, 31.5], [20.25, 11.75]]])
    dirs = np.concatenate([random_unit_dirs(9, 2, rng), unit_dirs_2d([0.0, math.pi / 2, math.pi / 4, math.pi, 1.25 * math.pi])])
    f = rng.uniform(0.05, 1.5, size=(32, 32, 8))
    act = np.repeat(np.repeat((lv >= 0).reshape(4, 4), 8, axis=0), 8, axis=1)
    f[~act] = 0.0
    i0 = rng.uniform(0, 2, size=(dirs.shape[0], 8))
    wl = iso_workload((32, 32), 8, f * 1.3, f, probes, dirs, active=act.astype(np.uint8), max_level=3, i0=i0)
    M = orc.build_mips(wl, max_level=3)
    M.levels = np.ascontiguousarray(lv[None, :])
    dw, grid, mips = _build(P, wl, max_level=3)
    mips.set_levels(M.levels)
    assert np.array_equal(mips.levels(), M.levels)
    _solve_and_compare(P, wl, M, dw, grid, mips)


def test_edge_cases(P):
    # no probes
    wl = make("C1", n=32, n_dirs=4)
    full = wl.probe_pos
    wl.probe_pos = full[:0]
    dw, grid, mips = _build(P, wl)
    J = P.pipeline.mean_intensity(dw, grid, mips)
    assert J.shape == (0, 8)
    # ragged probe count (not a multiple of any lane grouping), single direction
    wl.probe_pos = full[:37]
    wl.dirs, wl.weights = wl.dirs[:1], wl.weights[:1]
    M = orc.build_mips(wl)
    dw, grid, mips = _build(P, wl)
    _solve_and_compare(P, wl, M, dw, grid, mips)
    # all bricks empty: every intensity is exactly the (attenuation-free) boundary value
    wl2 = make("C2", n=64, n_dirs=4, n_probes=50)
    wl2.active[:] = 0
    wl2.eta[:] = 0
    wl2.chi[:] = 0
    wl2.i0 = np.full((4, wl2.n_lambda), 0.5, dtype=np.float32)
    dw, grid, mips = _build(P, wl2)
    assert grid.info()[1] == 0 and (mips.levels() == -1).all()
    I, cap = P.pipeline.formal_solution(dw, grid, mips, capture_batch=0)
    assert (cap.counts.cpu().numpy() == 0).all()
    assert (I.cpu().numpy() == 0.5).all()
    # capture overflow is reported, counts stay complete
    wl3 = make("C1", n=32, n_dirs=4, n_probes=10)
    M3 = orc.build_mips(wl3)
    res = orc.hdda_march(wl3, M3, capture_batch=0)
    dw, grid, mips = _build(P, wl3)
    with pytest.raises(P.DexError) as ei:
        P.pipeline.formal_solution(dw, grid, mips, capture_batch=0, want_I=False, room=3)
    assert ei.value.status == P.binding.DEX_ERR_CAPACITY
    # pure emitters (chi = 0, eta > 0: I_out = I_in + eta h ds) next to absorbing and to void cells
    rng = np.random.default_rng(12)
    chi = rng.uniform(0.0, 0.3, size=(64, 64, 8))
    eta = rng.uniform(0.0, 1.0, size=(64, 64, 8))
    chi[:, 20:40] = 0.0
    eta[30:50, 30:60] = 0.0
    chi[5:9, 5:9] = 1e-36           # far below 2^-60: treated as chi = 0 by the march records
    wl4 = iso_workload((64, 64), 16, eta, chi, rng.uniform(0, 64, size=(200, 2)), dirs_2d(12)[0], h=1.7)
    M4 = orc.build_mips(wl4)
    dw, grid, mips = _build(P, wl4)
    _solve_and_compare(P, wl4, M4, dw, grid, mips, lanes=(1, 8))
    # argument errors
    with pytest.raises(P.DexError):
        P.pipeline.build_mips(dw, grid, max_level=5)
    with pytest.raises(P.DexError):
        P.dex_build_sparse_grid(2, (64, 60), 16, 1.0)


def test_accuracy_regimes(P):
    """Thin (chi ~ 1e-6) and thick (chi ~ 30) media, long rays: the fp32 recurrence must hold 1e-5."""
    rng = np.random.default_rng(4)
    n = 512
    for scale in (1e-6, 1e-3, 0.3, 30.0):
        chi = scale * np.exp(rng.standard_normal((n, n, 8)))
        S = np.exp(0.5 * rng.standard_normal((n, n, 1)))
        probes = rng.uniform(0, n, size=(256, 2))
        wl = iso_workload((n, n), 16, chi * S, chi, probes, dirs_2d(8)[0])
        M = orc.build_mips(wl)
        dw, grid, mips = _build(P, wl)
        res = orc.hdda_march(wl, M)
        for lpr in (8, 1):
            P.dex_set_lanes_per_ray(lpr)
            I, _ = P.pipeline.formal_solution(dw, grid, mips)
            assert max_rel(I.cpu().numpy(), res.I) <= TOL, f"scale={scale}"
    P.dex_set_lanes_per_ray(1)


# ------------------------------------------------------------------------------------------ anisotropic
def _check_aux(P, wl, M, mips):
    act = orc.brick_active(wl)
    for m in range(M.max_level + 1):
        mask = _active_cell_mask(wl, act, m)
        vel = mips.level_data(P.DEX_CHAIN_VEL, m)
        nd = wl.ndim
        assert np.array_equal(vel[mask][:, :nd].view(np.uint32), np.ascontiguousarray(M.vbar[m])[mask].view(np.uint32))
        assert np.array_equal(vel[mask][:, 3].view(np.uint32), np.ascontiguousarray(M.vmax[m])[mask].view(np.uint32))
        line = mips.level_data(P.DEX_CHAIN_LINE, m)
        for l in range(wl.n_lines):
            for q, ref in enumerate((M.eta_star, M.chi_star, M.a0, M.inv_dlamD)):
                assert np.array_equal(line[mask][:, l, q].view(np.uint32),
                                      np.ascontiguousarray(ref[m][l])[mask].view(np.uint32))


@pytest.mark.parametrize("name,n,metric,thr,gate", [("C4", 128, 1, 0.3, -1.0), ("C5", 64, 0, 0.3, 0.02),
                                                    ("C5", 64, 1, 5.0, -1.0)])
def test_cav_small(P, name, n, metric, thr, gate):
    wl = make(name, n=n, n_dirs=8, n_probes=300)
    wl.metric, wl.thr_eta, wl.thr_chi, wl.tau_gate = metric, thr, thr, gate
    M = orc.build_mips(wl)
    assert M.levels.max() >= 2
    dw, grid, mips = _build(P, wl)
    _check_build(P, wl, M, grid, mips)
    _check_aux(P, wl, M, mips)
    _solve_and_compare(P, wl, M, dw, grid, mips, lanes=(8, 2))


@pytest.mark.parametrize("name,kw,thr,extra", [("C4", dict(n=128, n_dirs=8, n_probes=300), 0.3, "plain"),
                                                ("C4", dict(n=128, n_dirs=6, n_probes=200), 0.3, "caps+interval"),
                                                ("C4", dict(n=64, n_dirs=4, n_probes=150), 0.3, "25d"),
                                                ("C5", dict(n=64, n_dirs=8, n_probes=300), 5.0, "plain"),
                                                ("C5", dict(n=64, n_dirs=6, n_probes=200), 5.0, "caps+interval"),
                                                ("C4", dict(n=64, n_dirs=6, n_probes=100), 0.3, "classic"),
                                                ("C3", dict(n=128, n_dirs=8, n_probes=300), None, "plain")])
def test_memo_parity(P, name, kw, thr, extra):
    """Core-and-Voigt memoised per direction (tuning knob "memo": eta, chi evaluated once per (cell, direction,
    batch) into march records, then the ISO march) against the oracle and against the in-march evaluation: segment
    counts exact, I and J within 1e-5 of the oracle in both modes (and of each other); with the
    near-field cap + a radiance interval, 2.5D rays, the Classic variant, 8 lanes per ray, the direction split and the
    rebuild pipeline's wavelength windows."""
    from workloads.gen import dirs_25d
    wl = make(name, **kw)
    if thr is not None:
        wl.thr_eta = wl.thr_chi = thr
    nd = wl.dirs.shape[0]
    caps = None
    if extra == "25d":
        wl.dirs, wl.weights, wl.sin_incl = dirs_25d(3, 4)
        nd = wl.dirs.shape[0]
    wl.i0 = np.random.default_rng(21).uniform(0, 1, size=(nd, wl.n_lambda)).astype(np.float32)
    if extra == "caps+interval":
        caps = [6.0, 24.0]
        wl.interval = (2.0, 70.0)
    variant = orc.CLASSIC if extra == "classic" else None
    if variant is None:
        M = orc.build_mips(wl)
        ref = orc.hdda_march(wl, M, level_cap_t=caps)
        dw, grid, mips = _build(P, wl)
    else:
        ref = orc.plain_march(wl, variant=orc.CLASSIC)
        dw, grid, mips = _build(P, wl, variant=P.DEX_CLASSIC)
    mips.set_level_caps(caps)
    Jref = orc.mean_intensity(ref.I, wl.weights)
    out = {}
    try:
        for memo in (0, 1):
            P.dex_set_tuning("memo", memo)
            for lpr, split in ((1, 0), (8, 0), (1, 1)):
                P.dex_set_lanes_per_ray(lpr)
                P.dex_set_tuning("dir_split", split)
                seg = torch.zeros(1, dtype=torch.int64, device="cuda:0")
                I, _ = P.pipeline.formal_solution(dw, grid, mips, segment_count=seg)
                if variant is None:
                    assert int(seg.item()) == ref.segments
                assert max_rel(I.cpu().numpy(), ref.I) <= TOL, f"memo={memo} lanes={lpr}"
                J = P.pipeline.mean_intensity(dw, grid, mips)
                assert max_rel(J.cpu().numpy(), Jref) <= TOL, f"memo={memo} lanes={lpr} split={split}"
                out[(memo, lpr, split)] = J
            if variant is None and extra == "plain":      # wavelength windows of the rebuild pipeline (io_base != 0)
                P.dex_set_lanes_per_ray(1)
                P.dex_set_tuning("dir_split", 0)
                Jp, _ = P.pipeline.mean_intensity_pipelined(dw, grid, 2)
                assert torch.equal(Jp, out[(memo, 1, 0)])
        assert max_rel(out[(1, 1, 0)].cpu().numpy(), out[(0, 1, 0)].cpu().numpy()) <= TOL
        assert torch.equal(out[(1, 1, 0)], out[(1, 1, 1)])       # the direction split sums in the fused order
    finally:
        P.dex_set_tuning("memo", -1)
        P.dex_set_tuning("dir_split", -1)
        P.dex_set_lanes_per_ray(1)



def test_memo_budget_and_allocation_failure(P):
    """The memoised march's temporaries under pressure: a caller-set bound ("memo_budget_mb") far below the whole spectrum's
    records still takes the memoised path, in more groups of wavelength batches, with bit-identical J (batches are
    independent columns); a records allocation that fails is retried with half the batches; when not even one batch
    fits before anything was marched, the solve falls back to evaluating eta, chi in the ray loop -- the "memo" = 0
    path bit for bit -- instead of failing.  Which path ran is read off the library's launch counter."""
    wl = make("C4", n=128, n_dirs=6, n_probes=300)
    wl.thr_eta = wl.thr_chi = 0.3
    assert wl.n_batch >= 4
    dw, grid, mips = _build(P, wl)

    def run():
        c0 = P.dex_launch_count()
        seg = torch.zeros(1, dtype=torch.int64, device="cuda:0")
        J = P.pipeline.mean_intensity(dw, grid, mips, segment_count=seg)
        torch.cuda.synchronize()
        return J, int(seg.item()), P.dex_launch_count() - c0

    try:
        P.dex_set_tuning("memo", 0)
        J0, s0, n0 = run()
        P.dex_set_tuning("memo", 1)
        assert P.dex_last_march_mapping()["memo_batches_per_group"] == 0
        J1, s1, n1 = run()
        assert P.dex_last_march_mapping()["memo_batches_per_group"] == wl.n_batch
        assert s1 == s0 and n1 > n0                       # the records kernel is an extra launch
        assert max_rel(J1.cpu().numpy(), J0.cpu().numpy()) <= TOL
        P.dex_set_tuning("memo_budget_mb", 1)             # below one batch's records: one batch per group
        Jb, sb, nb = run()
        assert torch.equal(Jb, J1) and sb == s1 and nb >= n1 + wl.n_batch - 1
        assert P.dex_last_march_mapping()["memo_batches_per_group"] == 1
        P.dex_set_tuning("memo_budget_mb", 0)
        P.dex_set_tuning("memo_fail_allocs", 1)           # the whole-spectrum allocation fails once: two groups
        Jf, sf, nf = run()
        assert torch.equal(Jf, J1) and sf == s1 and n1 < nf < nb
        assert P.dex_last_march_mapping()["memo_batches_per_group"] == (wl.n_batch + 1) // 2
        P.dex_set_tuning("memo_fail_allocs", 1000)        # nothing can be allocated: in-march evaluation
        Jx, sx, nx = run()
        assert torch.equal(Jx, J0) and sx == s0 and nx == n0
        assert P.dex_last_march_mapping()["memo_batches_per_group"] == 0
    finally:
        P.dex_set_tuning("memo_fail_allocs", 0)
        P.dex_set_tuning("memo_budget_mb", 0)
        P.dex_set_tuning("memo", -1)

def test_classic_equals_plain_march(P):
    wl = make("C4", n=64, n_dirs=6, n_probes=100)
    A = orc.plain_march(wl, variant=orc.CLASSIC)
    dw, grid, mips = _build(P, wl, variant=P.DEX_CLASSIC)
    assert (mips.levels() <= 0).all()
    I, _ = P.pipeline.formal_solution(dw, grid, mips)
    assert max_rel(I.cpu().numpy(), A.I) <= TOL


def test_velinterp_small(P):
    wl = make("C3", n=256, n_dirs=8, n_probes=300)
    M = orc.build_mips(wl)
    assert M.levels.max() >= 1
    dw, grid, mips = _build(P, wl)
    _check_build(P, wl, M, grid, mips)
    _check_aux(P, wl, M, mips)
    act = orc.brick_active(wl)
    for m in range(M.max_level + 1):
        mask = _active_cell_mask(wl, act, m)
        got = mips.level_data(P.DEX_CHAIN_VTAB, m)[mask]
        ref = M.vtab[m][mask]
        assert max_rel(got, ref) <= 2e-6
    _solve_and_compare(P, wl, M, dw, grid, mips, lanes=(8, 2))


# ------------------------------------------------------------------------------------------ full size
def test_c2_full_size_sampled(P):
    """configs[1] at BASELINE size in the launch configuration bench.py times (fused J over all probes);
    the oracle computes a seeded sample of probes one by one."""
    wl = make("C2")
    M = orc.build_mips(wl)
    dw, grid, mips = _build(P, wl)
    _check_build(P, wl, M, grid, mips, spectra=False)
    seg = torch.zeros(1, dtype=torch.int64, device="cuda:0")
    J = P.pipeline.mean_intensity(dw, grid, mips, segment_count=seg).cpu().numpy()
    rng = np.random.default_rng(77)
    idx = np.sort(rng.choice(wl.probe_pos.shape[0], size=192, replace=False))
    res = orc.hdda_march(wl, M, probe_pos=wl.probe_pos[idx])
    Jref = orc.mean_intensity(res.I, wl.weights)
    assert max_rel(J[idx], Jref) <= TOL
    assert int(seg.item()) > 0
    assert np.isfinite(J).all() and (J >= 0).all()
    # visit lists and path lengths of the timed launch's traversal at 512^2: 32 seeded probes x all 64 directions, every
    # wavelength batch (each has its own level table), bit-exact against the oracle
    sel = np.sort(rng.choice(wl.probe_pos.shape[0], size=32, replace=False))
    wl.probe_pos = np.ascontiguousarray(wl.probe_pos[sel])
    dw.t["probe_pos"] = torch.from_numpy(wl.probe_pos).cuda()
    for b in range(wl.n_batch):
        ref = orc.hdda_march(wl, M, capture_batch=b)
        _, cap = P.pipeline.formal_solution(dw, grid, mips, capture_batch=b, want_I=False)
        _check_lists(cap, ref, cap.room)


def test_direction_split_bit_identical(P):
    """Small problems (fewer probes than one wave of blocks) are launched one block per (probe tile, batch, direction)
    into a temporary I and summed by the reduction kernel in the fused kernel's order: J and the segment count are bit
    for bit those of the fused launch, for every lanes-per-ray mapping, with boundary intensity; pool memory is returned
    by dex_trim."""
    wl = make("C2", n=128, n_dirs=12, n_probes=700)
    wl.i0 = np.random.default_rng(5).uniform(0, 1, size=(12, wl.n_lambda)).astype(np.float32)
    M = orc.build_mips(wl)
    ref = orc.hdda_march(wl, M)
    dw, grid, mips = _build(P, wl)
    try:
        for lpr in (1, 8):
            P.dex_set_lanes_per_ray(lpr)
            out = {}
            for split in (0, -1, 1, 5):
                P.dex_set_tuning("dir_split", split)
                seg = torch.zeros(1, dtype=torch.int64, device="cuda:0")
                out[split] = P.pipeline.mean_intensity(dw, grid, mips, segment_count=seg)
                assert int(seg.item()) == ref.segments
            assert max_rel(out[0].cpu().numpy(), orc.mean_intensity(ref.I, wl.weights)) <= TOL
            for split in (-1, 1, 5):
                assert torch.equal(out[0], out[split]), f"lanes={lpr} dir_split={split}"
    finally:
        P.dex_set_tuning("dir_split", -1)
        P.dex_set_lanes_per_ray(1)
    mips.destroy(); grid.destroy()
    torch.cuda.synchronize()
    assert P.dex_trim() >= 0


# ------------------------------------------------------------------------------------------ host entry
@pytest.mark.parametrize("name,kw", [("C2", dict(n=128, n_dirs=8, n_probes=333)), ("C5", dict(n=32, n_dirs=6, n_probes=200)),
                                     ("C3", dict(n=128, n_dirs=6, n_probes=150))])
def test_host_entry_matches_device_path(P, name, kw):
    """dex_mean_intensity_host (HOST buffers in, host J out: bench.py's e2e leg) gives bit for bit the J and the
    segment count of the three device-pointer calls it chains, with pinned and with pageable inputs."""
    wl = make(name, **kw)
    wl.i0 = np.random.default_rng(3).uniform(0, 1, size=(wl.dirs.shape[0], wl.n_lambda)).astype(np.float32)
    dw, grid, mips = _build(P, wl)
    seg = torch.zeros(1, dtype=torch.int64, device="cuda:0")
    J = P.pipeline.mean_intensity(dw, grid, mips, segment_count=seg).cpu().numpy()
    for pinned in (P.pipeline.pin(wl), None):
        Jh, nseg, h2d, d2h = P.pipeline.solve_J_from_host(wl, "cuda:0", pinned)
        assert nseg == int(seg.item()) and nseg > 0
        assert np.array_equal(Jh.view(np.uint32), J.view(np.uint32))
        assert d2h == J.size * 4 + 8 and 0 < h2d <= dw.h2d_bytes
    # the host entry uploads dense spectra: a wavelength stride is refused (it would read past the uploads)
    import paper_2511_08498_b200.binding as Bm
    orig = Bm._mips_desc

    def strided(*a, **k):
        d, n, keep = orig(*a, **k)
        d.lambda_stride = 2 * wl.n_lambda
        return d, n, keep
    Bm._mips_desc = strided
    try:
        with pytest.raises(P.DexError):
            P.pipeline.solve_J_from_host(wl, "cuda:0")
    finally:
        Bm._mips_desc = orig
    # argument errors surface as a status, not a crash
    with pytest.raises(P.DexError):
        P.dex_mean_intensity_host(2, (64, 60), 16, 1.0, None, dict(variant=0, n_lambda=8, lambda_batch=8, max_level=0,
                                  metric=1, thr_eta=0.0, thr_chi=0.0, tau_gate=-1.0,
                                  eta=torch.zeros(64 * 60 * 8), chi=torch.zeros(64 * 60 * 8)),
                                  P.Rays(torch.zeros(1, 2), torch.ones(1, 2), torch.ones(1)), torch.zeros(1, 8))


# ------------------------------------------------------------------------------------------ Voigt function
def test_voigt_profile_against_oracle(P):
    """H(a, x) as the Core-and-Voigt march evaluates it (dex_voigt_profile) against the oracle's HUM1WEI24
    (PAPER.md:329): the fp64 form to 1e-9, the fp32 table form (damping window of csrc/dex_voigt.cuh) to 1e-6,
    across the core, the wings, the region-I switch at |x| + a = 15 and far beyond it."""
    rng = np.random.default_rng(5)
    x = np.concatenate([rng.uniform(-15.5, 15.5, 200000), rng.uniform(-4, 4, 100000), [0.0, 14.99, 15.0, -15.0, 40.0, 3e3, -2e5],
                        np.arange(0, 481) / 32.0, (np.arange(0, 480) + 0.5) / 32.0])
    for a0 in (1e-4, 4.9e-3, 5e-3, 0.01, 0.02, 0.03, 0.031, 0.3, 2.0):
        a = np.full(x.shape, a0, dtype=np.float32)
        ref = orc.voigt_H(a.astype(np.float64), x)
        ta, tx = torch.from_numpy(a).cuda(), torch.from_numpy(x).cuda()
        # lanes whose |x| + a lies within rounding of the switch may take the other branch (5e-5 apart there)
        near = np.abs(np.abs(x) + a0 - 15.0) < 1e-5
        H64 = P.dex_voigt_profile(ta, tx, mode=1).cpu().numpy()
        assert max_rel(H64[~near], ref[~near]) <= 1e-9, f"a={a0}"
        H = P.dex_voigt_profile(ta, tx, mode=0).cpu().numpy()
        assert max_rel(H[~near], ref[~near]) <= 1e-6, f"a={a0}"
        assert max_rel(H[near], ref[near]) <= 1e-4


# ------------------------------------------------------------------------------------------ full size, C3-C5
def _crops(wl, rng, n_crops, side_bricks):
    """Seeded brick-aligned boxes that contain active bricks."""
    b, nd = wl.brick, wl.ndim
    act = orc.brick_active(wl)
    bd = wl.brick_dims
    out = []
    while len(out) < n_crops:
        lo_b = [int(rng.integers(0, bd[a] - side_bricks + 1)) for a in range(nd)]
        lo = [v * b for v in lo_b]
        size = [side_bricks * b] * nd
        ids = crop_brick_ids(wl, lo, size)
        if act[ids].any():
            out.append((lo, size, ids))
    return out


@pytest.mark.parametrize("name,side", [("C3", 6), ("C4", 6), ("C5", 3)])
def test_full_size_build_on_crops(P, name, side):
    """BASELINE-size builds (configs[2..4]): slot table exact over the whole grid; level table, packed words and
    every mip chain exact against the oracle on seeded crops (the build is brick-local, see crop_workload)."""
    wl = make(name, n_probes=64)
    dw, grid, mips = _build(P, wl)
    act = orc.brick_active(wl)
    slots = grid.slots()
    assert np.array_equal(slots >= 0, act)
    lv = mips.levels()
    assert ((lv >= 0) == act[None, :]).all()
    full = {}
    rng = np.random.default_rng(99)
    for lo, size, ids in _crops(wl, rng, 3, side):
        cw = crop_workload(wl, lo, size)
        Mc = orc.build_mips(cw)
        assert np.array_equal(lv[:, ids], Mc.levels), f"{name}: levels differ in the crop at {lo}"
        nd = wl.ndim
        for m in range(Mc.max_level + 1):
            sl = tuple(slice(lo[a] >> m, (lo[a] + size[a]) >> m) for a in reversed(range(nd)))
            mask = _active_cell_mask(cw, orc.brick_active(cw), m)
            for chain, ref in ((P.DEX_CHAIN_ETA, Mc.eta[m]), (P.DEX_CHAIN_CHI, Mc.chi[m])):
                if (chain, m) not in full:
                    full[(chain, m)] = mips.level_data(chain, m)
                got = full[(chain, m)][sl]
                assert np.array_equal(got[mask].view(np.uint32), np.ascontiguousarray(ref)[mask].view(np.uint32))
            if (P.DEX_CHAIN_VEL, m) not in full:
                full[(P.DEX_CHAIN_VEL, m)] = mips.level_data(P.DEX_CHAIN_VEL, m)
            vel = full[(P.DEX_CHAIN_VEL, m)][sl]
            assert np.array_equal(vel[mask][:, :nd].view(np.uint32), np.ascontiguousarray(Mc.vbar[m])[mask].view(np.uint32))
            assert np.array_equal(vel[mask][:, 3].view(np.uint32), np.ascontiguousarray(Mc.vmax[m])[mask].view(np.uint32))
            # the four mip chains per line: bit-exact
            if (P.DEX_CHAIN_LINE, m) not in full:
                full[(P.DEX_CHAIN_LINE, m)] = mips.level_data(P.DEX_CHAIN_LINE, m)
            line = full[(P.DEX_CHAIN_LINE, m)][sl]
            for l in range(wl.n_lines):
                for q, ref in enumerate((Mc.eta_star, Mc.chi_star, Mc.a0, Mc.inv_dlamD)):
                    assert np.array_equal(line[mask][:, l, q].view(np.uint32),
                                          np.ascontiguousarray(ref[m][l])[mask].view(np.uint32)), f"{name}: line chain {q}"
            # the velocity tables the C3 march reads (4 GB at level 0), every batch, every level: 2e-6 (DESIGN tolerances)
            if wl.variant == orc.VELINTERP:
                tab = mips.level_data(P.DEX_CHAIN_VTAB, m)[sl]
                assert max_rel(tab[mask], Mc.vtab[m][mask]) <= 2e-6, f"{name}: vtab level {m}"
                del tab
    hist = [int((lv == m).sum()) for m in range(-1, wl.max_level + 1)]
    assert sum(hist) == lv.size          # Table-2 style histogram covers every (batch, brick)


# wavelength batches whose oracle pyramid is built over the WHOLE grid (numpy, 3-26 s each): C3 far wing + line core;
# C4 core of the blended pair (two active lines), core of the 600 nm line (one), continuum (none); C5 line core
FULL_SIZE_BATCHES = {"C3": (0, 4), "C4": (3, 20, 25), "C5": (1,)}


@pytest.mark.parametrize("name", ["C3", "C4", "C5"])
def test_full_size_march_sampled(P, name):
    """BASELINE-size grids (configs[2..4]), the workload's own VLM variant, the launch bench.py times (fused J over all
    probes) against the ORACLE: for the batches of FULL_SIZE_BATCHES the oracle pyramid is built over the whole grid
    (batches are independent, batch_workload) -- level table and packed words exact over the whole grid, every mip
    chain of the batch bit-exact over the whole grid (velocity tables 2e-6), visit lists and path lengths bit-exact on
    32 seeded probes x all directions, I of those rays and J of those probes (from the all-probe fused launch) within
    1e-5.  Then (ii) the Classic (level 0, per-voxel velocity) march against the oracle's plain AW87 march."""
    wl = make(name)
    dw, grid, mips = _build(P, wl)
    all_probes = wl.probe_pos
    seg = torch.zeros(1, dtype=torch.int64, device="cuda:0")
    J_all = P.pipeline.mean_intensity(dw, grid, mips, segment_count=seg).cpu().numpy()
    assert int(seg.item()) > 0 and np.isfinite(J_all).all() and (J_all >= 0).all()
    lv = mips.levels()
    act = orc.brick_active(wl)
    rng = np.random.default_rng(31)
    idx = np.sort(rng.choice(all_probes.shape[0], size=32, replace=False))
    wl.probe_pos = np.ascontiguousarray(all_probes[idx])
    dw.t["probe_pos"] = torch.from_numpy(wl.probe_pos).cuda()
    I = P.pipeline.formal_solution(dw, grid, mips)[0].cpu().numpy()
    chains = {}
    for b in FULL_SIZE_BATCHES[name]:
        sub, lam_idx = batch_workload(wl, [b])
        Mb = orc.build_mips(sub)
        assert np.array_equal(lv[b], Mb.levels[0]), f"{name} batch {b}: {(lv[b] != Mb.levels[0]).sum()} brick levels differ"
        assert np.array_equal(mips.packed_levels(b), orc.pack_levels(Mb.levels[0], Mb.max_level))
        for m in range(Mb.max_level + 1):
            mask = _active_cell_mask(wl, act, m)
            for chain, ref in ((P.DEX_CHAIN_ETA, Mb.eta[m]), (P.DEX_CHAIN_CHI, Mb.chi[m])):
                if (chain, m) not in chains:
                    chains[(chain, m)] = mips.level_data(chain, m)
                got = np.ascontiguousarray(chains[(chain, m)][..., lam_idx])
                assert np.array_equal(got[mask].view(np.uint32), np.ascontiguousarray(ref)[mask].view(np.uint32))
            if wl.variant == orc.VELINTERP:
                tab = mips.level_data(P.DEX_CHAIN_VTAB, m)[mask][:, :, lam_idx]
                assert max_rel(tab, Mb.vtab[m][mask]) <= 2e-6, f"{name} batch {b}: vtab level {m}"
                del tab
        ref = orc.hdda_march(sub, Mb, capture_batch=0)
        _, cap = P.pipeline.formal_solution(dw, grid, mips, capture_batch=b, want_I=False)
        _check_lists(cap, ref, cap.room)
        del cap
        assert ref.segments > 0 and ref.counts.max() > 64        # long rays through several levels
        assert max_rel(I[:, :, lam_idx], ref.I) <= TOL, f"{name} batch {b}: I"
        assert max_rel(J_all[idx][:, lam_idx], orc.mean_intensity(ref.I, wl.weights)) <= TOL, f"{name} batch {b}: J"
    chains.clear()
    # (ii) exact side at full size against the oracle
    wl.probe_pos = np.ascontiguousarray(wl.probe_pos[:6 if name == "C4" else 24])
    dw.t["probe_pos"] = torch.from_numpy(wl.probe_pos).cuda()
    A = orc.plain_march(wl, variant=orc.CLASSIC)
    mc = P.pipeline.build_mips(dw, grid, variant=P.DEX_CLASSIC)
    Ic, _ = P.pipeline.formal_solution(dw, grid, mc)
    assert max_rel(Ic.cpu().numpy(), A.I) <= TOL
    Jc = P.pipeline.mean_intensity(dw, grid, mc).cpu().numpy()
    assert max_rel(Jc, orc.mean_intensity(A.I, wl.weights)) <= TOL


# ------------------------------------------------------------------------------------------ T8: near-field MIP cap
@pytest.mark.parametrize("name,kw,thr", [("C2", dict(n=256, n_dirs=12, n_probes=800), 0.05),
                                         ("C5", dict(n=64, n_dirs=8, n_probes=300), 5.0),
                                         ("C3", dict(n=256, n_dirs=8, n_probes=200), None)])
def test_level_cap_parity(P, name, kw, thr):
    """dex_mips_set_level_caps against the oracle's capped HDDA: visit lists and path lengths bit-exact, I and J within
    1e-5, for the paper-analogue thresholds (6, 24, 96, 384), a dense set of small thresholds, and the two limits."""
    wl = make(name, **kw)
    if thr is not None:
        wl.thr_eta = wl.thr_chi = thr
    M = orc.build_mips(wl)
    assert M.levels.max() >= 2
    dw, grid, mips = _build(P, wl)
    base = orc.hdda_march(wl, M, capture_batch=0)
    for caps in (orc.level_caps_paper(), [2.5, 5.0, 11.0, 40.0], [1e9, 1e9, 1e9, 1e9], []):
        mips.set_level_caps(caps)
        ref = orc.hdda_march(wl, M, capture_batch=0, level_cap_t=caps)
        _, cap = P.pipeline.formal_solution(dw, grid, mips, capture_batch=0, want_I=False)
        _check_lists(cap, ref, cap.room)
        seg = torch.zeros(1, dtype=torch.int64, device="cuda:0")
        I, _ = P.pipeline.formal_solution(dw, grid, mips, segment_count=seg)
        assert int(seg.item()) == ref.segments
        assert max_rel(I.cpu().numpy(), ref.I) <= TOL
        J = P.pipeline.mean_intensity(dw, grid, mips)
        assert max_rel(J.cpu().numpy(), orc.mean_intensity(ref.I, wl.weights)) <= TOL
        if len(caps) == 0:
            assert ref.segments == base.segments
    with pytest.raises(P.DexError):
        mips.set_level_caps([5.0, 2.0])


# ------------------------------------------------------------------------------------------ large coordinates
def _large_void_workload(n=4096, brick=16, seed=31):
    """A large, mostly empty 2D ISO medium: populated bricks in a few blobs and isolated single bricks, wide voids in
    between (empty-space distance up to the cap of 8 bricks), brick-constant eta, chi so that any level table is a
    valid one.  Probes anywhere (in voids, on voxel and brick planes); random, axis-parallel, diagonal and grazing
    directions.  Input recipe only."""
    rng = np.random.default_rng(seed)
    nb = n // brick
    yy, xx = np.mgrid[0:nb, 0:nb]
    occ = np.zeros((nb, nb), dtype=bool)
    for _ in range(14):
        cx, cy, r = rng.uniform(0, nb), rng.uniform(0, nb), rng.uniform(3, 22)
        occ |= (xx - cx) ** 2 + (yy - cy) ** 2 < r * r
    occ |= rng.random((nb, nb)) < 0.004                      # isolated bricks inside the voids
    occ[0, :] |= rng.random(nb) < 0.3                        # and some on the grid's edges and corners
    occ[:, -1] |= rng.random(nb) < 0.3
    occ[0, 0] = occ[-1, -1] = True
    val = rng.uniform(0.002, 0.02, size=(nb, nb)).astype(np.float32) * occ
    field = np.repeat(np.repeat(val, brick, axis=0), brick, axis=1)                    # [n][n] fp32
    spec = np.ascontiguousarray(np.repeat(field.reshape(-1, 1), 8, axis=1))            # [nvox][8]
    act = np.repeat(np.repeat(occ, brick, axis=0), brick, axis=1).astype(np.uint8).ravel()
    probes = np.concatenate([
        rng.uniform(0, n, size=(150, 2)),
        rng.integers(0, n, size=(20, 2)).astype(np.float64),                 # on voxel corners
        rng.integers(0, nb, size=(20, 2)).astype(np.float64) * brick,        # on brick corners
        rng.integers(0, n, size=(20, 2)) + 0.5,                              # voxel centres
        [[0.0, 0.0], [n - 0.001, n - 0.001], [n - 0.5, 0.5], [0.25, n - 0.25]]]).astype(np.float32)
    ang = np.array([0.0, math.pi / 2, math.pi, 1.5 * math.pi, math.pi / 4, 0.75 * math.pi, 1.25 * math.pi, 1.75 * math.pi,
                    1e-6, math.pi / 2 + 1e-5, math.pi - 3e-7, 1.5 * math.pi + 2e-4, math.atan2(1, 2), math.atan2(-3, 1)])
    dirs = np.concatenate([unit_dirs_2d(ang), random_unit_dirs(10, 2, rng)]).astype(np.float32)
    from workloads.gen import METRIC_RELVAR, VARIANT_ISO, Workload
    wl = Workload(name="large-void", ndim=2, dims=(n, n, 1), brick=brick, voxel_size=1.0, active=act, variant=VARIANT_ISO,
                  n_lambda=8, lambda_batch=8, max_level=4, metric=METRIC_RELVAR, thr_eta=1e-3, thr_chi=1e-3, tau_gate=-1.0,
                  probe_pos=np.ascontiguousarray(probes), dirs=np.ascontiguousarray(dirs),
                  weights=np.full(dirs.shape[0], 1.0 / dirs.shape[0], dtype=np.float32), eta=spec * np.float32(1.5), chi=spec)
    levels = np.where(occ.ravel(), rng.integers(0, 5, size=nb * nb), -1).astype(np.int8)[None, :]
    return wl, levels


def test_large_grid_void_boxes_list_parity(P):
    """Visit lists of the PRODUCTION traversal (cap-free crossing, whole boxes of empty bricks in one step, single-step
    fine-coordinate correction) against the oracle's HDDA on a 4096^2 grid that is ~80 % empty: bit-exact records and
    path lengths for 214 probes x 24 directions.  This is what holds dex_fine_coord to its claim that the fp32 position
    locates the T5 cell to within one voxel at large coordinates and over a whole-axis search: a guess two voxels off
    would enter a wrong cell or brick and change the list.  Repeated under a near-field cap (the other crossing routine)."""
    wl, levels = _large_void_workload()
    act_b = orc.brick_active(wl)
    assert 0.1 < act_b.mean() < 0.35
    M = orc.build_mips(wl, max_level=4)
    M.levels = np.ascontiguousarray(levels)
    dw, grid, mips = _build(P, wl, max_level=4)
    assert np.array_equal(grid.slots() >= 0, act_b)
    mips.set_levels(M.levels)
    for caps in ([], [6.0, 24.0, 96.0, 384.0]):
        mips.set_level_caps(caps)
        ref = orc.hdda_march(wl, M, capture_batch=0, level_cap_t=caps if caps else None)
        assert ref.segments > 100000
        _, cap = P.pipeline.formal_solution(dw, grid, mips, capture_batch=0, want_I=False)
        _check_lists(cap, ref, cap.room)
        seg = torch.zeros(1, dtype=torch.int64, device="cuda:0")
        J = P.pipeline.mean_intensity(dw, grid, mips, segment_count=seg)
        assert int(seg.item()) == ref.segments
        assert max_rel(J.cpu().numpy(), orc.mean_intensity(ref.I, wl.weights)) <= TOL


def test_velocity_bin_report(P):
    """dex_mips_velocity_bin_report against the oracle: per-line maximum ratio bit-exact, counts exact."""
    wl = make("C3", n=256, n_dirs=4, n_probes=16)
    dw, grid, mips = _build(P, wl)
    for factor in (2.0, 1.0, 0.25):
        mx, over = mips.velocity_bin_report(factor)
        rmx, rover = orc.velocity_bin_report(wl, factor)
        assert np.array_equal(mx.view(np.uint32), rmx.view(np.uint32)) and np.array_equal(over, rover)
    assert over[0] > 0
    wl2 = make("C4", n=64, n_dirs=4, n_probes=16)
    _, _, m2 = _build(P, wl2)
    with pytest.raises(P.DexError):
        m2.velocity_bin_report(2.0)


# ------------------------------------------------------------------------------------------ 2.5D rays (8(f)-2)
@pytest.mark.parametrize("name,kw", [("C2", dict(n=256, n_probes=600)), ("C4", dict(n=128, n_probes=200)),
                                     ("C3", dict(n=128, n_probes=150))])
def test_25d_rays_parity(P, name, kw):
    """dex_rays.d_sin_incl (PAPER.md:347 Gauss-Radau inclinations) against the oracle for the three providers: visit
    lists unchanged and bit-exact, I and J within 1e-5; also through the host entry; 3D grids reject it."""
    from workloads.gen import dirs_25d
    wl = make(name, n_dirs=4, **kw)
    if name == "C4":
        wl.thr_eta = wl.thr_chi = 0.3
    wl.dirs, wl.weights, wl.sin_incl = dirs_25d(5, 4)
    M = orc.build_mips(wl)
    dw, grid, mips = _build(P, wl)
    ref = _solve_and_compare(P, wl, M, dw, grid, mips, lanes=(1, 4))
    flat = orc.hdda_march(wl, M, sin_incl=np.ones(20, dtype=np.float32))
    assert max_rel(ref.I, flat.I) > 1e-3                     # the inclination changes the answer
    Jh, nseg, _, _ = P.pipeline.solve_J_from_host(wl, "cuda:0")
    assert nseg == ref.segments
    assert max_rel(Jh, orc.mean_intensity(ref.I, wl.weights)) <= TOL
    w3 = make("C5", n=32, n_dirs=4, n_probes=20)
    w3.sin_incl = np.ones(4, dtype=np.float32)
    d3, g3, m3 = _build(P, w3)
    with pytest.raises(P.DexError):
        P.pipeline.mean_intensity(d3, g3, m3)


# ------------------------------------------------------------------------------------------ T10: radiance intervals
@pytest.mark.parametrize("name,kw,thr", [("C2", dict(n=256, n_dirs=12, n_probes=700), 0.05),
                                         ("C5", dict(n=64, n_dirs=8, n_probes=300), 5.0)])
def test_radiance_interval_parity(P, name, kw, thr):
    """dex_rays.t_begin / t_end (Algorithm 1's HDDA(t1, t2)) against the oracle: clipped visit lists and path lengths
    bit-exact, I and J within 1e-5, with a boundary intensity entering at t_end and together with the near-field cap."""
    wl = make(name, **kw)
    wl.thr_eta = wl.thr_chi = thr
    wl.i0 = np.random.default_rng(9).uniform(0, 1, size=(wl.dirs.shape[0], wl.n_lambda)).astype(np.float32)
    M = orc.build_mips(wl)
    dw, grid, mips = _build(P, wl)
    for interval, caps in (((0.0, 7.5), None), ((6.0, 24.0), None), ((24.0, 96.0), [6.0, 24.0]), ((3.0, 1.0e9), None)):
        wl.interval = interval
        mips.set_level_caps(caps)
        ref = orc.hdda_march(wl, M, capture_batch=0, level_cap_t=caps)
        _, cap = P.pipeline.formal_solution(dw, grid, mips, capture_batch=0, want_I=False)
        _check_lists(cap, ref, cap.room)
        seg = torch.zeros(1, dtype=torch.int64, device="cuda:0")
        I, _ = P.pipeline.formal_solution(dw, grid, mips, segment_count=seg)
        assert int(seg.item()) == ref.segments
        assert max_rel(I.cpu().numpy(), ref.I) <= TOL
        J = P.pipeline.mean_intensity(dw, grid, mips)
        assert max_rel(J.cpu().numpy(), orc.mean_intensity(ref.I, wl.weights)) <= TOL
    wl.interval = (5.0, 2.0)
    with pytest.raises(P.DexError):
        P.pipeline.mean_intensity(dw, grid, mips)


# ------------------------------------------------------------------------------------------ 8(f)-3: rebuild pipeline
@pytest.mark.parametrize("name,kw,caps", [("C2", dict(n=256, n_dirs=12, n_probes=900), None),
                                          ("C2", dict(n=128, n_dirs=8, n_probes=300), [6.0, 24.0]),
                                          ("C3", dict(n=128, n_dirs=8, n_probes=300), None),
                                          ("C4", dict(n=128, n_dirs=8, n_probes=150), None),
                                          ("C5", dict(n=64, n_dirs=8, n_probes=300), None)])
def test_rebuild_pipeline_parity(P, name, kw, caps):
    """dex_mean_intensity_pipelined (mips of stage s+1 built on a second stream while stage s is marched, two stages
    resident) against the oracle: level table bit-exact, segment count exact, J within 1e-5; and against the
    whole-spectrum path of the library, bit for bit, for every stage size including a ragged last stage."""
    wl = make(name, **kw)
    wl.i0 = np.random.default_rng(11).uniform(0, 1, size=(wl.dirs.shape[0], wl.n_lambda)).astype(np.float32)
    M = orc.build_mips(wl)
    ref = orc.hdda_march(wl, M, level_cap_t=caps)
    Jref = orc.mean_intensity(ref.I, wl.weights)
    dw, grid, mips = _build(P, wl)
    mips.set_level_caps(caps)
    seg0 = torch.zeros(1, dtype=torch.int64, device="cuda:0")
    J0 = P.pipeline.mean_intensity(dw, grid, mips, segment_count=seg0)
    assert int(seg0.item()) == ref.segments
    for bps in sorted({1, 2, 3, wl.n_batch, wl.n_batch + 5}):
        seg = torch.zeros(1, dtype=torch.int64, device="cuda:0")
        J, lv = P.pipeline.mean_intensity_pipelined(dw, grid, bps, level_caps=caps, segment_count=seg, want_levels=True)
        torch.cuda.synchronize()
        assert np.array_equal(lv, M.levels), f"bps={bps}: level tables differ"
        assert int(seg.item()) == ref.segments
        assert max_rel(J.cpu().numpy(), Jref) <= TOL
        assert torch.equal(J, J0), f"bps={bps}: pipelined J differs from the whole-spectrum path"
    # a new iteration's eta (here: halved) goes through the same call, no handle surviving between the two
    if name == "C2":
        dw.t["eta"] = dw.t["eta"] * 0.5
        wl.eta = (wl.eta * np.float32(0.5)).astype(np.float32)
        J2, lv2 = P.pipeline.mean_intensity_pipelined(dw, grid, 2, level_caps=caps, want_levels=True)
        M2 = orc.build_mips(wl)
        assert np.array_equal(lv2, M2.levels)
        r2 = orc.hdda_march(wl, M2, level_cap_t=caps)
        assert max_rel(J2.cpu().numpy(), orc.mean_intensity(r2.I, wl.weights)) <= TOL
    with pytest.raises(P.DexError):
        P.pipeline.mean_intensity_pipelined(dw, grid, 0)


# ------------------------------------------------------------------------------------------ T11: single-direction VLM
@pytest.mark.parametrize("name,kw,thr,tilt", [("C4", dict(n=128, n_dirs=8, n_probes=200), 0.3, False),
                                              ("C4", dict(n=64, n_dirs=6, n_probes=120), 0.1, True),
                                              ("C5", dict(n=64, n_dirs=8, n_probes=300), 5.0, False)])
def test_single_direction_vlm_parity(P, name, kw, thr, tilt):
    """dex_direction_fields and dex_mean_intensity_single_direction against the oracle: direction fields
    within 2e-6 (fp64 Voigt, one fp32 rounding; exactly 0 in empty bricks), per-direction level tables bit-exact,
    segment count exact, J within 1e-5, with boundary intensity, the near-field cap and 2.5D rays."""
    wl = make(name, **kw)
    wl.thr_eta = wl.thr_chi = thr
    nd = wl.dirs.shape[0]
    wl.i0 = np.random.default_rng(13).uniform(0, 1, size=(nd, wl.n_lambda)).astype(np.float32)
    if tilt:
        wl.sin_incl = np.linspace(0.35, 1.0, nd).astype(np.float32)
    dw = P.pipeline.upload(wl, "cuda:0")
    grid = P.pipeline.build_grid(dw)
    for k in (0, nd // 2, nd - 1):
        e_ref, c_ref = orc.direction_fields(wl, wl.dirs[k], None if wl.sin_incl is None else wl.sin_incl[k])
        e, c = P.pipeline.direction_fields(dw, grid, k)
        e, c = e.cpu().numpy(), c.cpu().numpy()
        assert max_rel(e, e_ref) <= 2e-6 and max_rel(c, c_ref) <= 2e-6
        assert np.array_equal(e == 0, e_ref == 0) and np.array_equal(c == 0, c_ref == 0)
    for caps in (None, [6.0, 24.0]):
        Jref, lv_ref, seg_ref = orc.single_direction_solve(wl, level_cap_t=caps)
        seg = torch.zeros(1, dtype=torch.int64, device="cuda:0")
        J, lv = P.pipeline.mean_intensity_single_direction(dw, grid, level_caps=caps, segment_count=seg, want_levels=True)
        assert np.array_equal(lv, lv_ref), f"level tables differ in {(lv != lv_ref).sum()} entries"
        assert (lv_ref > 0).any()
        assert int(seg.item()) == seg_ref
        assert max_rel(J.cpu().numpy(), Jref) <= TOL
    # the all-in-one call is the chain of its building blocks: fields -> ISO mips -> one-direction march, accumulated
    J2 = torch.zeros_like(J)
    for k in range(nd):
        e, c = P.pipeline.direction_fields(dw, grid, k)
        m = P.dex_build_vlm_mips(grid, P.DEX_ISO, wl.n_lambda, wl.lambda_batch, wl.max_level, wl.metric, wl.thr_eta,
                                 wl.thr_chi, wl.tau_gate, eta=e, chi=c)
        m.set_level_caps([6.0, 24.0])
        t = dw.t
        r = P.Rays(t["probe_pos"], t["dirs"][k:k + 1].contiguous(), t["weights"][k:k + 1].contiguous(),
                   t["i0"][k:k + 1].contiguous(), None if wl.sin_incl is None else t["sin_incl"][k:k + 1].contiguous())
        Jk = torch.empty_like(J)
        P.dex_mean_intensity(grid, m, r, Jk)
        J2 += Jk
        m.destroy()
    assert max_rel(J2.cpu().numpy(), J.cpu().numpy()) <= 2e-6
    with pytest.raises(P.DexError):       # a static medium has no direction dependence
        P.pipeline.mean_intensity_single_direction(dw, grid, variant=P.DEX_ISO)


def test_edge_cases_pipelined_and_single_direction(P):
    """Degenerate inputs of the two composite entries: no probes, one batch (a single stage), all bricks empty, no
    directions; argument errors."""
    # no probes: nothing to write, the level table is still built and returned
    wl = make("C2", n=64, n_dirs=4, n_probes=20)
    full = wl.probe_pos
    wl.probe_pos = full[:0]
    M = orc.build_mips(wl)
    dw = P.pipeline.upload(wl, "cuda:0")
    grid = P.pipeline.build_grid(dw)
    J, lv = P.pipeline.mean_intensity_pipelined(dw, grid, 1, want_levels=True)
    assert J.shape == (0, wl.n_lambda) and np.array_equal(lv, M.levels)
    # all bricks empty, boundary intensity only: J = sum_k w_k i0[k] exactly as the whole-spectrum path gives it
    wl2 = make("C2", n=64, n_dirs=4, n_probes=33)
    wl2.active[:] = 0
    wl2.eta[:] = 0
    wl2.chi[:] = 0
    wl2.i0 = np.random.default_rng(3).uniform(0, 1, size=(4, wl2.n_lambda)).astype(np.float32)
    dw2, g2, m2 = _build(P, wl2)
    J0 = P.pipeline.mean_intensity(dw2, g2, m2)
    seg = torch.zeros(1, dtype=torch.int64, device="cuda:0")
    J1, lv1 = P.pipeline.mean_intensity_pipelined(dw2, g2, 3, segment_count=seg, want_levels=True)
    assert torch.equal(J0, J1) and (lv1 == -1).all() and int(seg.item()) == 0
    assert max_rel(J1.cpu().numpy(), orc.mean_intensity(np.broadcast_to(wl2.i0, (33,) + wl2.i0.shape), wl2.weights)) <= 1e-6
    # single direction: no directions -> J = 0 (and overwritten, not added to); no probes -> no-op
    wl3 = make("C4", n=64, n_dirs=4, n_probes=25)
    dw3 = P.pipeline.upload(wl3, "cuda:0")
    g3 = P.pipeline.build_grid(dw3)
    J3 = torch.full((25, wl3.n_lambda), 7.0, dtype=torch.float32, device="cuda:0")
    r0 = P.Rays(dw3.t["probe_pos"], dw3.t["dirs"][:0], dw3.t["weights"][:0])
    P.dex_mean_intensity_single_direction(g3, P.pipeline._mips_args(wl3, dw3.t), r0, J3)
    assert (J3 == 0).all()
    # ... and a second call overwrites the first (J is not accumulated across calls)
    Ja, _ = P.pipeline.mean_intensity_single_direction(dw3, g3)
    Jb, _ = P.pipeline.mean_intensity_single_direction(dw3, g3, J=Ja.clone())
    assert torch.equal(Ja, Jb)
    rn = P.Rays(dw3.t["probe_pos"][:0], dw3.t["dirs"], dw3.t["weights"])
    P.dex_mean_intensity_single_direction(g3, P.pipeline._mips_args(wl3, dw3.t), rn,
                                          torch.empty((0, wl3.n_lambda), dtype=torch.float32, device="cuda:0"))
    # argument errors: max_level beyond log2(brick) is refused by both
    with pytest.raises(P.DexError):
        P.pipeline.mean_intensity_pipelined(dw, grid, 1, max_level=5)
    with pytest.raises(P.DexError):
        P.pipeline.mean_intensity_single_direction(dw3, g3, max_level=5)
