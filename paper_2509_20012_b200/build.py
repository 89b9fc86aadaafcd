"""Build the C-ABI CUDA library in-tree for sm_100a (nvcc cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libfredopt.so")
SOURCES = [os.path.join(CSRC, f) for f in ("plan_build.cu", "iterate.cu", "passes.cu", "no_alloc.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("fredopt_kernels.cuh", "kernels_iter.cuh", "kernels_eval.cuh", "fredopt_plan.cuh")] + \
    [os.path.join(os.path.dirname(HERE), "include", "fredopt.h")]


def nvcc_path() -> str:
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc"):
        if p and os.path.exists(p):
            return p
    return "nvcc"


def build_library(force: bool = False, verbose: bool = False, defines=()) -> str:
    """defines: extra -D... flags (the compile-time tunables of csrc/fredopt_kernels.cuh, e.g. -DFWD_U1=8; timing experiments
    such as -DEXP_NO_GATHER give wrong results on purpose).  A build with defines always recompiles."""
    if not force and not defines and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    cmd = [nvcc_path(), "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "--threads", "0",
           "-Xcompiler", "-fPIC", "-shared", "-o", LIB] + list(defines) + SOURCES
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
        print(" ".join(cmd), file=sys.stderr)
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build_library(force="--force" in sys.argv, verbose="-v" in sys.argv, defines=[a for a in sys.argv[1:] if a.startswith("-D")]))
