"""Build step: compile paper_1005_5384_b200/csrc into libtc_b200.so with nvcc for sm_100a.

In-tree, explicit nvcc (no JIT cache): the .so travels with the repository
snapshot to the GPU box.  Usable as ``python -m paper_1005_5384_b200.build``.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtc_b200.so")
SOURCES = ["tc_api.cpp", "tc_build.cpp", "tc_kernels.cu", "tc_kernels_dense.cu", "tc_build_gpu.cu", "tc_shard.cu"]
HEADERS = ["tc_internal.h", "tc_lanes.h", os.path.join("..", "..", "include", "tc.h"), os.path.join("..", "..", "include", "tc_bench.h")]

NVCC_FLAGS = [
    "-std=c++17", "-O3", "-lineinfo",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-Xcompiler", "-fPIC,-fopenmp,-ffp-contract=off",
    "-Xptxas", "-v",
]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile the library if missing or older than its sources; return its path."""
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + ["-shared", "-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES] + ["-lgomp"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed building libtc_b200.so")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
