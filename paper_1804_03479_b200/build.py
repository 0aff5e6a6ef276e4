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
# translation units -> the headers each depends on (a unit is recompiled when one of them is newer than its object)
COMMON = ["mhd_physics.cuh", "mhd_eigen.cuh", "mhd_recon.cuh", "mhd_kernels.cuh", "mhd_kernels2.cuh", "mhd_kernels3.cuh",
          "mhd_ctu_pass1.cuh", "mhd_vl_pass1.cuh", "mhd_march.h"]
UNITS = {
    "mhd_api.cu": COMMON + ["mhd_api_host.inl", "mhd_api_grid.inl", "mhd_api_amr.inl", "mhd_grid.cuh", "mhd_amr.cuh", "mhd_prolong.cuh",
                            os.path.join("..", "..", "include", "mhd.h")],
    "mhd_march.cu": COMMON + ["mhd_vl_march.cuh"],
    "mhd_noalloc.cu": ["mhd_physics.cuh", "mhd_eigen.cuh", "mhd_recon.cuh", "mhd_kernels.cuh", "mhd_kernels2.cuh", "mhd_kernels3.cuh",
                       os.path.join("..", "..", "include", "mhd.h")],
}
OBJDIR = os.path.join(HERE, "build")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr",
]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def _newer(paths, t) -> bool:
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in paths)


def _build_lib(lib: str, tag: str, extra, force: bool, verbose: bool) -> str:
    """compile the stale translation units (in parallel) into build/<tag>_<unit>.o and link them into `lib`"""
    os.makedirs(OBJDIR, exist_ok=True)
    objs, procs = [], []
    for src, deps in UNITS.items():
        obj = os.path.join(OBJDIR, f"{tag}_{os.path.splitext(src)[0]}.o")
        objs.append(obj)
        if force or not os.path.exists(obj) or _newer([src] + deps, os.path.getmtime(obj)):
            cmd = [nvcc()] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + \
                  (["--split-compile", "0"] if src == "mhd_api.cu" else []) + ["-c", os.path.join(CSRC, src), "-o", obj]
            procs.append((cmd, subprocess.Popen(cmd)))
    for cmd, pr in procs:
        if pr.wait() != 0:
            raise subprocess.CalledProcessError(pr.returncode, cmd)
    if procs or not os.path.exists(lib) or any(os.path.getmtime(o) > os.path.getmtime(lib) for o in objs):
        subprocess.check_call([nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a"] + objs + ["-o", lib])
    return lib


def build(force: bool = False, verbose: bool = False) -> str:
    return _build_lib(LIB, "std", [], force, verbose)


LIB_IEEE32 = os.path.join(HERE, "libmhd_ieee32.so")


def build_ieee32(force: bool = False) -> str:
    """Control build for tests/fp32_controls.py only (never loaded by the product path unless MHD_LIBPATH points at it):
    the same sources with -DMHD_IEEE32, i.e. IEEE-rounded FP32 division / square root instead of the SFU approximations."""
    return _build_lib(LIB_IEEE32, "ieee32", ["-DMHD_IEEE32"], force, False)


def build_variant(tag: str, defines, force: bool = False) -> str:
    """A/B builds for experiments: the same sources with extra -D switches -> libmhd_<tag>.so (load it with MHD_LIBPATH)"""
    return _build_lib(os.path.join(HERE, f"libmhd_{tag}.so"), tag, list(defines), force, False)


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
    if "--variant" in sys.argv:
        k = sys.argv.index("--variant")
        print(build_variant(sys.argv[k + 1], [a for a in sys.argv[k + 2:] if a.startswith("-D")], force="--force" in sys.argv))
    if "--ieee32" in sys.argv:
        print(build_ieee32(force="--force" in sys.argv))
