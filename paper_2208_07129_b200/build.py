"""Build the C-ABI shared library in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2208_07129_b200.build [--force] [--verbose]

Produces paper_2208_07129_b200/csrc/libfe_mf.so (git-ignored; it travels with gpurun snapshots) and, beside it,
libfe_chfsi.so (include/fe_chfsi.h: the subspace iteration around the operator; links libfe_mf.so, cuBLAS, cuSOLVER).
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(CSRC, "libfe_mf.so")
SOURCES = ["fe_mf.cu", "fe_probe.cu"]
DEPS = ["fe_kernels.cuh", "fe_kernels_eo.cuh", "fe_kernels_cart2.cuh", "fe_kernels_tma.cuh", "fe_kernels_gen.cuh", "fe_kernels_plane.cuh", "fe_kernels_line.cuh", "fe_kernels_kron.cuh", "fe_kernels_oi.cuh", "fe_init_ahead.cuh", "fe_tables.h", "fe_dispatch.inl", os.path.join("..", "..", "include", "fe_mf.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "--fmad=true",
    "-Xcompiler", "-fPIC,-O2",
    "-shared",
]


LIB_CHFSI = os.path.join(CSRC, "libfe_chfsi.so")
CHFSI_SOURCES = ["fe_chfsi.cu"]
CHFSI_DEPS = [os.path.join("..", "..", "include", "fe_chfsi.h"), os.path.join("..", "..", "include", "fe_mf.h")]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA library cannot be built (there is no CPU fallback)")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    for f in SOURCES + DEPS:
        path = os.path.join(CSRC, f)
        if os.path.exists(path) and os.path.getmtime(path) > t:
            return True
    return False


def _stale(lib: str, files) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.exists(os.path.join(CSRC, f)) and os.path.getmtime(os.path.join(CSRC, f)) > t for f in files)


def build_chfsi(force: bool = False, verbose: bool = False) -> str:
    """libfe_chfsi.so; a separate library so that libfe_mf.so itself depends on nothing but the CUDA runtime."""
    build(force=False, verbose=verbose)
    if not force and not _stale(LIB_CHFSI, CHFSI_SOURCES + CHFSI_DEPS) and os.path.getmtime(LIB_CHFSI) >= os.path.getmtime(LIB):
        return LIB_CHFSI
    nvcc = nvcc_path()
    cuda_lib = os.path.join(os.path.dirname(os.path.dirname(os.path.realpath(nvcc))), "lib64")
    cmd = [nvcc] + NVCC_FLAGS + [os.path.join(CSRC, s) for s in CHFSI_SOURCES] + \
          ["-o", LIB_CHFSI, "-L" + CSRC, "-lfe_mf", "-lcublas", "-lcusolver",
           "-Xlinker", "-rpath=$ORIGIN", "-Xlinker", "-rpath=" + cuda_lib]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(" ".join(cmd) + "\n" + res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libfe_chfsi.so")
    return LIB_CHFSI


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    cmd = [nvcc_path()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
          [os.path.join(CSRC, s) for s in SOURCES if os.path.exists(os.path.join(CSRC, s))] + ["-o", LIB]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(" ".join(cmd) + "\n" + res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libfe_mf.so")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
    print(build_chfsi(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
