"""Builds the C-ABI shared library in-tree: paper_2104_10000_b200/liblandau_b200.so (sm_100a only).

Each source is compiled to an object under paper_2104_10000_b200/build/ (git-ignored), in parallel and only
when it or a header changed, then linked.  `python -m paper_2104_10000_b200.build` forces a full rebuild and
prints the register / shared-memory usage of every kernel (-Xptxas -v)."""
from __future__ import annotations

import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "liblandau_b200.so")
OBJ = os.path.join(HERE, "build")
SOURCES = ["landau_setup.cpp", "landau_kernels.cu", "landau_shared.cu", "landau_band.cu", "landau_api.cu"]
HEADERS = ["landau_internal.h", "landau_kernels.h", "landau_launch.cuh", "landau_pair_math.cuh", os.path.join(ROOT, "include", "landau.h")]


def _hdr_time() -> float:
    return max(os.path.getmtime(h if os.path.isabs(h) else os.path.join(HERE, "csrc", h)) for h in HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = os.environ.get("LANDAU_NVCC_FLAGS", "").split()   # e.g. -DPAIR_MIN_BLOCKS=6 for tuning sweeps
    base = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC",
            "-I", os.path.join(ROOT, "include"), "-I", os.path.join(HERE, "csrc")] + extra
    if verbose:
        base += ["-Xptxas", "-v"]
    os.makedirs(OBJ, exist_ok=True)
    flags_file = os.path.join(OBJ, "flags.txt")
    flags = " ".join(base)
    if not os.path.exists(flags_file) or open(flags_file).read() != flags:
        force = True
    hdr_t = _hdr_time()
    jobs = []
    for s in SOURCES:
        src = os.path.join(HERE, "csrc", s)
        obj = os.path.join(OBJ, os.path.splitext(s)[0] + ".o")
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(src), hdr_t):
            jobs.append(base + ["-c", src, "-o", obj])
    if jobs:
        with ThreadPoolExecutor(max_workers=len(jobs)) as ex:
            list(ex.map(subprocess.check_call, jobs))
        open(flags_file, "w").write(flags)
    objs = [os.path.join(OBJ, os.path.splitext(s)[0] + ".o") for s in SOURCES]
    if jobs or not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(o) for o in objs):
        subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB] + objs)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
