"""Builds paper_1502_07478_b200/libjpet.so (the C-ABI of include/jpet.h) with nvcc for sm_100a, in-tree.

The tiled event kernel is instantiated once per group of shapes (csrc/rows_inst.cu with -DJPET_GROUP=g); the groups
and csrc/jpet_api.cu are compiled in parallel into paper_1502_07478_b200/build/*.o and linked into the library.
"""
from __future__ import annotations

import concurrent.futures
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
OBJ = os.path.join(_HERE, "build")
LIB = os.path.join(_HERE, "libjpet.so")
N_GROUPS = 4
HEADERS = [os.path.join(CSRC, f) for f in ("common.cuh", "image_kernels.cuh", "sort_kernels.cuh", "histogram.cuh", "generator.cuh",
                                           "mlem_rows.cuh", "mlem_direct.cuh", "rows_launch.h", "task_table.h")] + [
    os.path.join(os.path.dirname(_HERE), "include", "jpet.h")]
# (object, source, extra flags)
UNITS = [("jpet_api.o", "jpet_api.cu", [])] + [(f"rows_inst_{g}.o", "rows_inst.cu", [f"-DJPET_GROUP={g}"]) for g in range(N_GROUPS)]
DEPS = HEADERS + [os.path.join(CSRC, "jpet_api.cu"), os.path.join(CSRC, "rows_inst.cu")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--use_fast_math",
              "-Xcompiler", "-fPIC"]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _stale(target: str, deps) -> bool:
    return not os.path.exists(target) or any(os.path.getmtime(target) < os.path.getmtime(d) for d in deps)


def _compile(unit, verbose: bool) -> str:
    obj, src, extra = unit
    out = os.path.join(OBJ, obj)
    cmd = [nvcc_path(), *NVCC_FLAGS, *extra, *(["-Xptxas", "-v"] if verbose else []), "-c", "-o", out, os.path.join(CSRC, src)]
    subprocess.run(cmd, check=True)
    return out


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile what is missing or older than a source; returns the path of the library."""
    if not force and not _stale(LIB, DEPS):
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    todo = [u for u in UNITS if force or _stale(os.path.join(OBJ, u[0]), HEADERS + [os.path.join(CSRC, u[1])])]
    with concurrent.futures.ThreadPoolExecutor(max_workers=min(len(UNITS), os.cpu_count() or 1)) as pool:
        list(pool.map(lambda u: _compile(u, verbose), todo))
    subprocess.run([nvcc_path(), "-shared", "-o", LIB, *[os.path.join(OBJ, u[0]) for u in UNITS]], check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
