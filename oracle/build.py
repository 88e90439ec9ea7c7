"""Build the CPU oracle (TEST INFRASTRUCTURE) with gcc: oracle/liboracle.so (fp64) and
oracle/liboracle_f32.so (fp32 diagnostic mode).  No CUDA, nothing shared with the product."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "orc.c")
LIB64 = os.path.join(HERE, "liboracle.so")
LIB32 = os.path.join(HERE, "liboracle_f32.so")


def _stale(lib):
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(os.path.join(HERE, s)) > t for s in ("orc.c", "orc.h"))


def build(force: bool = False) -> None:
    base = ["gcc", "-O3", "-ffp-contract=off", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-fno-fast-math", SRC, "-lm"]
    for lib, extra in ((LIB64, []), (LIB32, ["-DORC_REAL_FLOAT"])):
        if force or _stale(lib):
            subprocess.check_call(base + extra + ["-o", lib])


if __name__ == "__main__":
    build(force=True)
    print("built", LIB64, LIB32)
