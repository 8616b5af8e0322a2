"""Build libhqmc.so (hand-written CUDA, sm_100a only) in-tree with nvcc."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libhqmc.so")
SOURCES = ["hqmc.cu", "hqmc_noalloc.cu"]      # hqmc_noalloc.cu: self-contained (the allocation-free S_B entry point)
HEADER = os.path.join("..", "..", "include", "hqmc.h")


def deps():
    """Every header / include file of csrc (the single translation unit hqmc.cu includes them all) and the public header."""
    return [f for f in sorted(os.listdir(CSRC)) if f.endswith((".cuh", ".h", ".inl"))] + [HEADER]


NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC",
              "-shared", "--expt-relaxed-constexpr", "-cudart", "static",
              "-lcufft", "-Xlinker", "-rpath=/usr/local/cuda/lib64"]      # cuFFT: the FFT of Eq.19 (library primitive)


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + deps())


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
