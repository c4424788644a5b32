"""Compile the CUDA sources in csrc/ for sm_100a into paper_2511_08498_b200/libdex.so (in-tree)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdex.so")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC", "-Xcompiler", "-fno-fast-math"]
# per-file extra flags: the build kernels' fp64 statistics must not be FMA-contracted (DESIGN.md V-rules)
SOURCES = {
    "dex_api.cu": [],
    "grid_build.cu": [],
    "grid_static.cu": [],
    "mips_build.cu": ["-fmad=false"],
    "march.cu": [],
    "peaks.cu": [],
}


def _newer(target, deps):
    if not os.path.exists(target):
        return False
    t = os.path.getmtime(target)
    return all(os.path.getmtime(d) <= t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    # DEX_NVCC_EXTRA: extra nvcc flags (e.g. -DDEX_MARCH_MINB=7) for tuning experiments; forces a rebuild
    extra_env = os.environ.get("DEX_NVCC_EXTRA", "").split()
    force = force or bool(extra_env)
    headers = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    headers.append(os.path.join(os.path.dirname(HERE), "include", "dex.h"))
    objs = []
    for src, extra in SOURCES.items():
        s = os.path.join(CSRC, src)
        o = os.path.join(CSRC, src.replace(".cu", ".o"))
        objs.append(o)
        if force or not _newer(o, [s] + headers):
            cmd = ["nvcc"] + ARCH + COMMON + extra + extra_env + (["-Xptxas", "-v"] if verbose else []) + ["-c", s, "-o", o]
            subprocess.run(cmd, check=True)
    if force or not _newer(LIB, objs):
        subprocess.run(["nvcc"] + ARCH + ["-shared", "-o", LIB] + objs + ["-lcudart"], check=True)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
