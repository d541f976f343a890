"""Compile the C oracle into oracle/liboracle.so.  TEST INFRASTRUCTURE (see oracle.h).

Usage: python -m oracle.build    (also called by __graft_entry__.build() and tests/conftest.py)
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["scan_hist.c", "chain_f32.c", "jacobi.c", "gemm_gelu.c", "image.c", "sssp.c", "sobel.c"]
LIB = os.path.join(HERE, "liboracle.so")


def build(force: bool = False) -> str:
    srcs = [os.path.join(HERE, s) for s in SOURCES]
    deps = srcs + [os.path.join(HERE, "oracle.h")]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    # -ffp-contract=off: reading C1-1 (no FMA contraction).  Plain -O2, single-threaded, no -march.
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-std=c11", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-o", LIB] + srcs + ["-lm"]
    subprocess.check_call(cmd, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
