"""In-tree build of the C-ABI CUDA library (nvcc, sm_100a only).

`python -m paper_2006_06866_b200.build` or `build()` compiles csrc/gce_ce.cu (host code, C ABI, the small kernels) and
csrc/gce_search_family.cu once per kernel family and mode (-DGCE_FAMILY=<n_phi> -DGCE_DUMP=<0|1>: the k_search
instantiations) into objects in a scratch directory, in parallel, and links them into paper_2006_06866_b200/libgce_ce.so.
nvcc cross-compiles without a GPU.  -fmad=false is part of the arithmetic contract: a
contracted multiply-add would change phase-bin indices; every translation unit gets it.
"""
from __future__ import annotations

import hashlib
import os
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
HDR = os.path.join(ROOT, "include", "gce_ce.h")
LIB = os.path.join(HERE, "libgce_ce.so")
OBJ_DIR = os.path.join(HERE, "build")

FAMILIES = (0, 15, 20, 30, 50)   # compile-time n_phi of the k_search families (0 = generic)
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17", "-fmad=false",
    "-Xcompiler", "-fPIC",
    "-I", os.path.join(ROOT, "include"),
]


def _units():
    """(object name, source, extra flags) of every translation unit."""
    units = [("gce_ce.o", os.path.join(CSRC, "gce_ce.cu"), [])]
    for n in FAMILIES:
        for d in (0, 1):
            units.append((f"gce_search_n{n}_d{d}.o", os.path.join(CSRC, "gce_search_family.cu"),
                          [f"-DGCE_FAMILY={n}", f"-DGCE_DUMP={d}"]))
    return units


def _deps():
    return [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith((".cu", ".cuh")) and f != "gce_ablation.cu"] + [HDR, os.path.abspath(__file__)]


def _code_only(text: str) -> str:
    """C / C++ source with comments and blank space removed, so that editing documentation does not change the hash."""
    import re
    text = re.sub(r"/\*.*?\*/", " ", text, flags=re.S)
    text = re.sub(r"//[^\n]*", " ", text)
    return " ".join(text.split())


def source_hash() -> str:
    """SHA-256 over what the library's code is built from -- the csrc files and the header without their comments, the
    compiler flags and the family list (bench.py ties ncu-derived numbers to it)."""
    h = hashlib.sha256()
    for p in _deps():
        if p.endswith(".py"):
            continue
        with open(p, "r") as f:
            h.update(_code_only(f.read()).encode())
    h.update(repr((NVCC_FLAGS[:-1], FAMILIES)).encode())   # the last flag is the include path of this checkout
    return h.hexdigest()[:16]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(p) > t for p in _deps())


def build(force: bool = False, verbose: bool = False, extra_flags=(), jobs: int | None = None) -> str:
    if not (force or _stale()):
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    tag = f".tmp{os.getpid()}"
    obj_dir = OBJ_DIR + tag   # private to this process: concurrent builds (ranks, test workers) do not collide
    os.makedirs(obj_dir, exist_ok=True)

    def compile_unit(u):
        name, src, flags = u
        obj = os.path.join(obj_dir, name)
        cmd = [nvcc, *NVCC_FLAGS, *extra_flags, *flags, *(["-Xptxas", "-v"] if verbose else []), "-c", "-o", obj, src]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on {name}:\n{r.stdout}\n{r.stderr}")
        if verbose:
            sys.stderr.write(f"==== {name}\n{r.stderr}\n")
        return obj

    objs = []
    try:
        with ThreadPoolExecutor(max_workers=jobs or os.cpu_count() or 4) as ex:
            objs = list(ex.map(compile_unit, _units()))
        tmp = LIB + tag
        subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", tmp, *objs])
        os.replace(tmp, LIB)
    finally:
        shutil.rmtree(obj_dir, ignore_errors=True)
    return LIB


ABLATION_LIB = os.path.join(HERE, "libgce_ablation.so")


def build_ablation(force: bool = False) -> str:
    """The design-ablation probe (csrc/gce_ablation.cu: the north_star's warp-per-trial + match_any histogram), its own
    shared object: bench.py --ablation and its GPU test load it; the product library does not contain it."""
    src = os.path.join(CSRC, "gce_ablation.cu")
    if not force and os.path.exists(ABLATION_LIB) and os.path.getmtime(ABLATION_LIB) >= os.path.getmtime(src):
        return ABLATION_LIB
    tmp = ABLATION_LIB + f".tmp{os.getpid()}"
    subprocess.check_call([os.environ.get("NVCC", "nvcc"), *NVCC_FLAGS, "-shared", "-o", tmp, src])
    os.replace(tmp, ABLATION_LIB)
    return ABLATION_LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
