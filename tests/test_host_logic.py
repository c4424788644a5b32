"""CPU-side checks of the product's host logic (no GPU, no compute calls through the library):

  * libdex.so builds, loads and exports every function include/dex.h declares;
  * the binding's EXPORTS list is the header's function list;
  * the multi-GPU sharding helpers (paper_2511_08498_b200/shard.py) on a world of 2 `gloo` ranks: probe ranges tile
    the probe list, the per-rank J rows all-gather into the single-rank result, job totals are max / sum over ranks.
"""
import ctypes
import importlib.util
import os
import re
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "dex.h")


def _lib_path():
    spec = importlib.util.spec_from_file_location("_dex_lib_build", os.path.join(ROOT, "paper_2511_08498_b200", "_build.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod.build()


def _declared_functions():
    """Names of the functions include/dex.h declares (comments stripped, `name(` at declaration level)."""
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", " ", src, flags=re.S)
    src = re.sub(r"//[^\n]*", " ", src)
    names = re.findall(r"\b(dex_[a-z0-9_]+)\s*\(", src)
    return sorted(set(names))


def test_header_declares_the_four_north_star_calls():
    names = _declared_functions()
    for n in ("dex_build_sparse_grid", "dex_build_vlm_mips", "dex_formal_solution", "dex_mean_intensity"):
        assert n in names


def test_library_exports_every_declared_symbol():
    lib = ctypes.CDLL(_lib_path())
    missing = [n for n in _declared_functions() if not hasattr(lib, n)]
    assert not missing, f"libdex.so lacks {missing}"
    lib.dex_version.restype = ctypes.c_char_p
    assert lib.dex_version()


def test_binding_names_match_header():
    _lib_path()
    from paper_2511_08498_b200 import binding
    assert sorted(binding.EXPORTS) == _declared_functions()


def test_compute_call_without_device_fails_loudly():
    """No CPU fallback: without a CUDA device a build call returns an error status, it does not compute."""
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    _lib_path()
    import paper_2511_08498_b200 as P
    with pytest.raises(P.DexError):
        P.dex_build_sparse_grid(2, (64, 64), 16, 1.0)


def test_lanes_query_sees_the_wavelength_count():
    """dex_get_lanes_per_ray is the host-side rule of the launch: a small problem is split over directions (2 lanes per
    ray) only while its temporary I of n_probes x n_dirs x n_lambda floats stays within 64 Mi floats; a problem of one
    wave of blocks or more runs one thread per ray.  Before any march the recorded mapping is all zero."""
    _lib_path()
    import paper_2511_08498_b200 as P
    P.dex_set_lanes_per_ray(0)
    try:
        assert P.dex_get_lanes_per_ray(4096, 16, 8) == 2
        assert P.dex_get_lanes_per_ray(4096, 16, 2048) == 8      # 128 Mi floats of I: not split, 8 lanes per ray
        assert P.dex_get_lanes_per_ray(1 << 20, 16, 8) == 1
        P.dex_set_lanes_per_ray(4)
        assert P.dex_get_lanes_per_ray(4096, 16, 8) == 4
    finally:
        P.dex_set_lanes_per_ray(0)
    if not torch.cuda.is_available():
        assert P.dex_last_march_mapping() == {"lanes_per_ray": 0, "dirs_per_block": 0, "memo_batches_per_group": 0}


# ------------------------------------------------------------------------------------------ sharding
def test_probe_ranges_tile_the_list():
    _lib_path()
    from paper_2511_08498_b200 import shard
    for n in (0, 1, 31, 32, 33, 1000, 262144, 262145):
        for world in (1, 2, 3, 8):
            spans = [shard.probe_range(n, world, r) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            for (a, b), (c, d) in zip(spans, spans[1:]):
                assert b == c and a <= b
            for lo, hi in spans[:-1]:
                assert lo % 32 == 0 and hi % 32 == 0 or hi == n
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) < 64
    with pytest.raises(ValueError):
        shard.probe_range(10, 2, 2)
    assert shard.rank_seed(8498002, 3) == 8498002 + 3000


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _rank_main(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import sys
        sys.path.insert(0, ROOT)
        from oracle import oracle as orc
        from paper_2511_08498_b200 import shard
        from workloads import make
        # "probes" mode: one atmosphere replicated, probe list cut into warp-aligned ranges, one all-gather of J
        wl = make("C2", n=64, n_dirs=4, n_probes=150)
        M = orc.build_mips(wl)
        lo, hi = shard.probe_range(wl.probe_pos.shape[0], world, rank)
        res = orc.hdda_march(wl, M, probe_pos=wl.probe_pos[lo:hi])
        J_local = torch.from_numpy(orc.mean_intensity(res.I, wl.weights))
        J = shard.gather_J(J_local, wl.probe_pos.shape[0])
        # "atmospheres" mode bookkeeping: max of the times, sum of the units
        ms, units = shard.job_totals(10.0 + rank, float(res.segments))
        seg_all = torch.tensor([float(res.segments)], dtype=torch.float64)
        dist.all_reduce(seg_all)
        np.save(os.path.join(out_dir, f"J_{rank}.npy"), J.numpy())
        np.save(os.path.join(out_dir, f"tot_{rank}.npy"), np.array([ms, units, float(seg_all.item()), lo, hi]))
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_probe_sharding(tmp_path):
    _lib_path()
    world = 2
    mp.spawn(_rank_main, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    from oracle import oracle as orc
    from workloads import make
    wl = make("C2", n=64, n_dirs=4, n_probes=150)
    M = orc.build_mips(wl)
    res = orc.hdda_march(wl, M)
    J_one = orc.mean_intensity(res.I, wl.weights)
    tots = [np.load(tmp_path / f"tot_{r}.npy") for r in range(world)]
    for r in range(world):
        J = np.load(tmp_path / f"J_{r}.npy")
        assert J.shape == J_one.shape
        assert np.array_equal(J, J_one), "all-gathered J differs from the single-rank J"
        assert tots[r][0] == 11.0                       # max over ranks of (10, 11)
        assert tots[r][1] == tots[r][2] == float(res.segments)
    assert tots[0][3] == 0 and tots[0][4] == tots[1][3] and tots[1][4] == 150


def test_crop_workload_is_brick_local():
    """tests/_util.crop_workload (used by the full-size GPU build tests): the oracle build of a brick-aligned crop
    equals the oracle build of the whole grid restricted to the crop's bricks."""
    from oracle import oracle as orc
    from workloads import make
    from _util import crop_brick_ids, crop_workload
    for name, n, lo, size in (("C4", 128, (32, 48), (64, 48)), ("C5", 32, (8, 0, 16), (16, 24, 16))):
        wl = make(name, n=n, n_dirs=4, n_probes=4)
        wl.thr_eta = wl.thr_chi = 0.3
        M = orc.build_mips(wl)
        cw = crop_workload(wl, lo, size)
        Mc = orc.build_mips(cw)
        ids = crop_brick_ids(wl, lo, size)
        assert np.array_equal(M.levels[:, ids], Mc.levels)
        for m in range(M.max_level + 1):
            sl = tuple(slice(lo[a] >> m, (lo[a] + size[a]) >> m) for a in reversed(range(wl.ndim)))
            assert np.array_equal(M.eta[m][sl], Mc.eta[m]) and np.array_equal(M.vmax[m][sl], Mc.vmax[m])


def test_batch_workload_is_a_column_selection():
    """workloads.gen.batch_workload (full-size GPU comparisons, bench.py's cpu_baseline): the oracle's level table and I
    of a workload restricted to some wavelength batches are the rows / columns of the full workload's, bit for bit."""
    from oracle import oracle as orc
    from workloads import make
    from workloads.gen import batch_workload
    for name, kw, batches in (("C2", dict(n=64, n_dirs=4, n_probes=40), [1, 3]), ("C4", dict(n=64, n_dirs=4, n_probes=30), [3, 20, 25]),
                              ("C3", dict(n=64, n_dirs=4, n_probes=30), [0, 4])):
        wl = make(name, **kw)
        wl.i0 = np.random.default_rng(2).uniform(0, 1, size=(4, wl.n_lambda)).astype(np.float32)
        M = orc.build_mips(wl)
        full = orc.hdda_march(wl, M)
        sub, idx = batch_workload(wl, batches)
        assert sub.n_lambda == 8 * len(batches) and sub.n_batch == len(batches)
        Ms = orc.build_mips(sub)
        assert np.array_equal(Ms.levels, M.levels[batches])
        part = orc.hdda_march(sub, Ms)
        assert np.array_equal(part.I, full.I[:, :, idx])


def test_bench_reference_arm_line():
    """bench.py --impl reference (the oracle on the host cores): one JSON line with the contract's keys."""
    import json
    import subprocess
    import sys
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "C1", "--steps", "1",
                          "--warmup", "0", "--cpu-probes", "64"], capture_output=True, text=True, timeout=600, check=True).stdout
    line = [ln for ln in out.splitlines() if ln.startswith("{")]
    assert len(line) == 1
    d = json.loads(line[0])
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e", "gpu_launches"):
        assert key in d, key
    assert d["impl"] == "reference" and d["value"] > 0 and d["gpu_launches"] == 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["cpu_baseline"]["kind"] == "oracle" and "workload" in d["config"]
