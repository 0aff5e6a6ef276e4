"""Build libmhd.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1804_03479_b200.build [--force]

The .so is git-ignored; it travels to the GPU box with the gpurun snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmhd.so")
SOURCES = ["mhd_api.cu"]
DEPS = ["mhd_api.cu", "mhd_api_host.inl", "mhd_api_grid.inl", "mhd_api_amr.inl", "mhd_physics.cuh", "mhd_eigen.cuh",
        "mhd_recon.cuh", "mhd_kernels.cuh", "mhd_kernels2.cuh", "mhd_kernels3.cuh", "mhd_grid.cuh", "mhd_amr.cuh", "mhd_prolong.cuh", "mhd_ctu_pass1.cuh", "mhd_vl_pass1.cuh",
        os.path.join("..", "..", "include", "mhd.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared", "--expt-relaxed-constexpr", "--split-compile", "0",
]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def stale(lib: str = LIB) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        cmd = [nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
              [os.path.join(CSRC, s) for s in SOURCES] + ["-o", LIB]
        subprocess.check_call(cmd)
    return LIB


LIB_IEEE32 = os.path.join(HERE, "libmhd_ieee32.so")


def build_ieee32(force: bool = False) -> str:
    """Control build for tests/fp32_controls.py only (never loaded by the product path unless MHD_LIBPATH points at it):
    the same sources with -DMHD_IEEE32, i.e. IEEE-rounded FP32 division / square root instead of the SFU approximations."""
    if force or stale(LIB_IEEE32):
        cmd = [nvcc()] + NVCC_FLAGS + ["-DMHD_IEEE32"] + [os.path.join(CSRC, s) for s in SOURCES] + ["-o", LIB_IEEE32]
        subprocess.check_call(cmd)
    return LIB_IEEE32


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
    if "--ieee32" in sys.argv:
        print(build_ieee32(force="--force" in sys.argv))
