"""Build liblpc.so (the C-ABI CUDA library) in-tree for sm_100a.

    python -m paper_2603_22553_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The library links cudart statically and
resolves cuTensorMapEncodeTiled at run time through cudaGetDriverEntryPoint,
so it needs neither libcuda at link time nor torch at any time.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liblpc.so")
SOURCES = [os.path.join(CSRC, "lpc_api.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("lpc_internal.cuh", "lpc_step.cuh", "lpc_step_vec.cuh", "lpc_step2.cuh", "lpc_precompute.cuh", "lpc_equil.cuh", "lpc_regions.cuh")] + [
    os.path.join(os.path.dirname(HERE), "include", "lpc.h")]

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared", "--extended-lambda",
]


def nvcc() -> str:
    cand = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "bin", "nvcc")
    return cand if os.path.exists(cand) else "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = [nvcc(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", tmp, *SOURCES]
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
