"""Builds the C-ABI shared library in-tree: paper_2104_10000_b200/liblandau_b200.so (sm_100a only)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "liblandau_b200.so")
SOURCES = ["landau_setup.cpp", "landau_kernels.cu", "landau_band.cu", "landau_api.cu"]
HEADERS = ["landau_internal.h", "landau_kernels.h", os.path.join(ROOT, "include", "landau.h")]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(HERE, "csrc", s) for s in SOURCES] + [h if os.path.isabs(h) else os.path.join(HERE, "csrc", h) for h in HEADERS]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
           "-Xcompiler", "-fPIC", "-shared", "-I", os.path.join(ROOT, "include"), "-I", os.path.join(HERE, "csrc")]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += os.environ.get("LANDAU_NVCC_FLAGS", "").split()   # e.g. -DPAIR_MIN_BLOCKS=6 for tuning sweeps
    cmd += [os.path.join(HERE, "csrc", s) for s in SOURCES] + ["-o", LIB]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
