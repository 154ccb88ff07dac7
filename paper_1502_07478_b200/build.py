"""Builds paper_1502_07478_b200/libjpet.so (the C-ABI of include/jpet.h) with nvcc for sm_100a, in-tree."""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libjpet.so")
SOURCES = [os.path.join(CSRC, "jpet_api.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("mlem_kernels.cuh", "mlem_rows2.cuh", "mlem_rows3.cuh", "task_table.h")] + [
    os.path.join(os.path.dirname(_HERE), "include", "jpet.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--use_fast_math",
              "-Xcompiler", "-fPIC", "-shared"]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile if the library is missing or older than any source; returns its path."""
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    cmd = [nvcc_path(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", LIB, *SOURCES]
    subprocess.run(cmd, check=True)
    return LIB


def build_microbench() -> str:
    """Roofline micro-benchmarks (FFMA, MUFU, red.global.add.f32, shared-memory RMW): csrc/microbench.cu -> csrc/microbench."""
    out = os.path.join(CSRC, "microbench")
    subprocess.run([nvcc_path(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-o", out,
                    os.path.join(CSRC, "microbench.cu")], check=True)
    return out


if __name__ == "__main__":
    if "--microbench" in sys.argv:
        print(build_microbench())
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
