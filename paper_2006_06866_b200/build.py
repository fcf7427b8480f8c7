"""In-tree build of the C-ABI CUDA library (nvcc, sm_100a only).

`python -m paper_2006_06866_b200.build` or `build()` compiles csrc/gce_ce.cu (one translation unit that includes
csrc/gce_*.cuh) into
paper_2006_06866_b200/libgce_ce.so.  nvcc cross-compiles without a GPU.  -fmad=false is part of the
arithmetic contract: a contracted multiply-add would change phase-bin indices.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
SRC = os.path.join(HERE, "csrc", "gce_ce.cu")
HDR = os.path.join(ROOT, "include", "gce_ce.h")
LIB = os.path.join(HERE, "libgce_ce.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17", "-fmad=false",
    "-Xcompiler", "-fPIC", "-shared",
    "-I", os.path.join(ROOT, "include"),
]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    csrc = os.path.dirname(SRC)
    deps = [os.path.join(csrc, f) for f in os.listdir(csrc) if f.endswith((".cu", ".cuh"))]
    return any(os.path.getmtime(p) > t for p in (*deps, HDR, os.path.abspath(__file__)))


def build(force: bool = False, verbose: bool = False, extra_flags=()) -> str:
    if force or _stale():
        nvcc = os.environ.get("NVCC", "nvcc")
        tmp = LIB + f".tmp{os.getpid()}"
        cmd = [nvcc, *NVCC_FLAGS, *extra_flags, *(["-Xptxas", "-v"] if verbose else []), "-o", tmp, SRC]
        subprocess.check_call(cmd)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
