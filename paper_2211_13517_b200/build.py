"""Builds the in-tree native libraries with nvcc for sm_100a.

  libfdas.so      the product: C ABI of include/fdas.h (K1 whitening, K2 fused convolution,
                  K3 harmonic sum, plan-time host mathematics, cuFFT R2C)

nvcc cross-compiles without a GPU.  Run ``python -m paper_2211_13517_b200.build``.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libfdas.so")
CUDA_HOME = os.environ.get("CUDA_HOME", "/usr/local/cuda")
NVCC = os.path.join(CUDA_HOME, "bin", "nvcc")

ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC"]

LIB_SOURCES = ["fdas_api.cu", "fdas_batch.cu", "fdas_convolve.cu", "fdas_convolve_tc.cu", "fdas_whiten.cu", "fdas_harmonic.cu", "fdas_host.cpp"]
HEADERS = ["fdas_fft_core.cuh", "fdas_tc_common.h", "fdas_host.h", "fdas_kernels.h", "fdas_maxcode.h", "fdas_plan_priv.h", os.path.join("..", "..", "include", "fdas.h")]


def _stale(target: str, sources) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    deps = [os.path.join(CSRC, s) for s in list(sources) + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def _run(cmd, verbose):
    if verbose:
        print(" ".join(cmd), flush=True)
    subprocess.run(cmd, check=True, cwd=CSRC)


def build_lib(force: bool = False, verbose: bool = False, ptxas_v: bool = False) -> str:
    if force or _stale(LIB, LIB_SOURCES):
        cmd = [NVCC] + ARCH + COMMON + (["-Xptxas", "-v"] if ptxas_v else []) + [
            "-shared", "-o", LIB] + LIB_SOURCES + [
            "-L" + os.path.join(CUDA_HOME, "lib64"), "-lcufft",
            "-Xlinker", "-rpath," + os.path.join(CUDA_HOME, "lib64")]
        _run(cmd, verbose)
    return LIB


def build_all(force: bool = False, verbose: bool = False):
    return build_lib(force, verbose)


if __name__ == "__main__":
    build_all(force="--force" in sys.argv, verbose=True)
