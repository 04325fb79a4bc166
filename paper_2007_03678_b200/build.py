"""Compile the CUDA library (csrc/adock.cu -> libadock.so, in-tree) for sm_100a with nvcc."""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libadock.so")
SOURCES = ["adock.cu"]
DEPS = ["adock.cu", "device.cuh", "lane.cuh", "lane_image.hpp", "topology.hpp", os.path.join("..", "..", "include", "adock.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-ftz=true",
              "-Xcompiler", "-fPIC", "-shared"]


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc, *NVCC_FLAGS, *os.environ.get("ADOCK_NVCC_EXTRA", "").split(), *(["-Xptxas", "-v"] if verbose else []), "-o", LIB,
               *[os.path.join(CSRC, s) for s in SOURCES]]
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
