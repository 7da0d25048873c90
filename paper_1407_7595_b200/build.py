"""In-tree build of the CUDA library (sm_100a only): `python -m paper_1407_7595_b200.build`.

nvcc cross-compiles without a GPU.  The .so lands beside this file so that it travels with a
snapshot of the repository; it is git-ignored.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmem_b200.so")
SOURCES = [os.path.join(CSRC, "mem_api.cu")]
HEADERS = [os.path.join(CSRC, f) for f in ("mem_common.cuh", "mem_processes.cuh", "mem_kernels.cuh", "mem_parton.cuh", "mem_tth.cuh")] + [
    os.path.join(ROOT, "include", "mem.h"), os.path.join(ROOT, "include", "mem_bench.h")]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in SOURCES + HEADERS + [os.path.abspath(__file__)])


def build(force: bool = False, verbose: bool = False) -> str:
    if force or is_stale():
        tmp = LIB + ".%d.tmp" % os.getpid()
        cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SOURCES
        subprocess.check_call(cmd)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
