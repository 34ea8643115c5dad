"""Build libsc_riccati.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsc_riccati.so")
SOURCES = ["sc_api.cu", "sc_static.cu"]
DEPS = ["sc_api.cu", "sc_static.cu", "sc_kernels.cuh", "sc_math.cuh", "sc_geometry.hpp", "sc_field_kernels.cuh", "sc_lowrank.cuh", "sc_probe_kernels.cuh",
        os.path.join("..", "..", "include", "sc_riccati.h")]


def nvcc_command(extra=()):
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    return [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
            "-Xcompiler", "-fPIC", "-shared", *extra,
            *[os.path.join(CSRC, s) for s in SOURCES], "-o", LIB, "-lcufft", "-lcusolver", "-lcublas",
            "-Xlinker", "-rpath=/usr/local/cuda/lib64"]


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        cmd = nvcc_command(("-Xptxas", "-v") if verbose else ())
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in __import__("sys").argv))
