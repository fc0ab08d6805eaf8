"""Build libkvpool.so (C ABI of include/kvpool.h) in-tree with nvcc for sm_100a.

    python -m paper_2606_14779_b200.build [--force]

The .so is git-ignored but travels to the GPU box with the gpurun snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libkvpool.so")
SOURCES = ["kvpool_core.cu", "kvpool_xfer.cu", "kvpool_dev.cu", "kvpool_ssd.cu", "kvpool_static.cu", "kernels.cu", "placement.cpp", "pool_mem.cpp", "ssd_io.cpp"]
HEADERS = ["kvpool_internal.hpp", "kernels.cuh", "placement.hpp", "pool_mem.hpp", "ssd_io.hpp", os.path.join("..", "..", "include", "kvpool.h"),
           os.path.join("..", "..", "include", "kvpool_dev.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--shared",
              "-Xcompiler", "-fPIC,-Wall,-Wextra,-fvisibility=hidden,-pthread", "-cudart", "shared"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = LIB + f".{os.getpid()}.tmp"
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + [os.path.join(CSRC, f) for f in SOURCES]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
