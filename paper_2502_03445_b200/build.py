"""Builds libtqc.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libtqc.so")
SOURCES = ["tqc_api.cu", "plan.cpp", "partition.cpp"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-ldl"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    deps.append(os.path.join(os.path.dirname(_HERE), "include", "tqc.h"))
    return any(os.path.getmtime(d) > t for d in deps)


PEAKS_LIB = os.path.join(_HERE, "libtqc_peaks.so")


def build_peaks(force: bool = False) -> str:
    """The measurement micro-benchmarks (csrc/peaks.cu -> libtqc_peaks.so); not loaded by the product path."""
    src = os.path.join(CSRC, "peaks.cu")
    if force or not os.path.exists(PEAKS_LIB) or os.path.getmtime(src) > os.path.getmtime(PEAKS_LIB):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
                               "-Xcompiler", "-fPIC", "-shared", "-o", PEAKS_LIB, src])
    return PEAKS_LIB


def build(force: bool = False, verbose: bool = False) -> str:
    build_peaks(force)
    if force or _stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        develop = ["-DTQC_DEVELOP"] if os.environ.get("TQC_DEVELOP") else []     # measurement switches
        cmd = [nvcc] + NVCC_FLAGS + develop + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + \
              [os.path.join(CSRC, s) for s in SOURCES]
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
