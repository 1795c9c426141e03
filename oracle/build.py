"""Build the CPU oracle (TEST INFRASTRUCTURE, not the product) into oracle/libcfs_oracle.so.

    python oracle/build.py

Flags: -O2 -ffp-contract=off so that the only fused multiply-adds are the explicit
fmaf() calls of cfs_oracle.c.  No CUDA, no code shared
with paper_2606_02226_b200/.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "cfs_oracle.c")
HDR = os.path.join(HERE, "cfs_oracle.h")
LIB = os.path.join(HERE, "libcfs_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB):
        newest = max(os.path.getmtime(SRC), os.path.getmtime(HDR))
        if os.path.getmtime(LIB) >= newest:
            return LIB
    cmd = ["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fno-fast-math", "-Wall", "-Wextra",
           "-shared", "-fPIC", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
