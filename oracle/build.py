"""Compile the CPU oracle (oracle/dex_oracle.c) into oracle/libdex_oracle.so.

Test infrastructure only.  No fast-math, no FMA contraction (the traversal contract is
stated op by op: SURVEY.md 8(c) T-rules); -mfma only makes the explicit fmaf() calls fast.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "dex_oracle.c")
LIB = os.path.join(HERE, "libdex_oracle.so")


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-std=gnu11", "-ffp-contract=off", "-fno-fast-math", "-mfma", "-fopenmp",
           "-shared", "-fPIC", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
