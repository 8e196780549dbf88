"""Builds tests/emu/libfdas_emu.so: the TEST-ONLY host emulator of the K2 / K2-TC CTAs (fdas_emu.cu)
together with the library's plan-time host mathematics.  Host code only (nvcc is used because the
sources share __host__ __device__ headers with the kernels)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(os.path.dirname(os.path.dirname(HERE)), "paper_2211_13517_b200", "csrc")
EMU = os.path.join(HERE, "libfdas_emu.so")
NVCC = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "bin", "nvcc")
SOURCES = [os.path.join(HERE, "fdas_emu.cu"), os.path.join(CSRC, "fdas_host.cpp")]
DEPS = SOURCES + [os.path.join(CSRC, h) for h in ("fdas_fft_core.cuh", "fdas_tc_common.h", "fdas_host.h", "fdas_maxcode.h")]


def build_emu(force: bool = False, verbose: bool = False) -> str:
    stale = not os.path.exists(EMU) or any(os.path.getmtime(d) > os.path.getmtime(EMU) for d in DEPS)
    if force or stale:
        cmd = [NVCC, "-O2", "-std=c++17", "-Xcompiler", "-fPIC", "-Wno-deprecated-gpu-targets", "-shared",
               "-o", EMU] + SOURCES
        if verbose:
            print(" ".join(cmd), flush=True)
        subprocess.run(cmd, check=True)
    return EMU


if __name__ == "__main__":
    build_emu(force=True, verbose=True)
