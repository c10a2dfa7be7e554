"""Builds libfdemri.so (the CUDA library behind include/fdemri.h) in-tree with nvcc for sm_100a."""
from __future__ import annotations

import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libfdemri.so")
SOURCES = ["fdemri.cu"]
DEPS = ["fdemri.cu", "fdemri_common.cuh", "fdemri_map.cuh", "fdemri_splines.cuh", "fdemri_sum.cuh", "fdemri_td.cuh", "fdemri_select.cuh", "airy_tables.inc", "poly_tables.inc", os.path.join("..", "..", "include", "fdemri.h")]

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "--fmad=true"]


def nvcc_path() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libfdemri cannot be built (there is no CPU fallback)")


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False, extra=()) -> str:
    if force or is_stale():
        extra = list(extra) + os.environ.get("FDEMRI_NVCC_EXTRA", "").split()
        cmd = [nvcc_path(), *NVCC_FLAGS, *extra, "-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
        if verbose:
            cmd.insert(1, "-Xptxas")
            cmd.insert(2, "-v")
        r = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
        if verbose:
            print(r.stdout, r.stderr)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + r.stdout + r.stderr)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
