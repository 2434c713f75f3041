"""Build the C-ABI shared library in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2208_07129_b200.build [--force] [--verbose]

Produces paper_2208_07129_b200/csrc/libfe_mf.so (git-ignored; it travels with gpurun snapshots) and, beside it,
libfe_chfsi.so (include/fe_chfsi.h: the subspace iteration around the operator; links libfe_mf.so, cuBLAS, cuSOLVER).
libfe_mf.so is several translation units (one per kernel family, fe_tu_*.cu, plus the host code and the constraint
matrices of include/fe_constraints.h) compiled in parallel and linked without relocatable device code.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(CSRC, "libfe_mf.so")
FE_MF_H = os.path.join("..", "..", "include", "fe_mf.h")
HOST_DEPS = ["fe_ctx.h", "fe_params.h", FE_MF_H]
KERNEL_DEPS = HOST_DEPS + ["fe_kernels.cuh", "fe_kernels_eo.cuh", "fe_kernels_cart2.cuh", "fe_kernels_tma.cuh"]
# translation unit -> the files it depends on (besides itself)
UNITS = {
    "fe_mf.cu": HOST_DEPS + ["fe_tables.h", "fe_eo_tables.h", "fe_oi_tables.h"],
    "fe_dispatch.cu": HOST_DEPS,
    "fe_probe.cu": [FE_MF_H],
    "fe_constraints.cu": [os.path.join("..", "..", "include", "fe_constraints.h"), FE_MF_H],
    "fe_tu_misc.cu": KERNEL_DEPS + ["fe_kernels_stream.cuh"],
    "fe_tu_gen.cu": KERNEL_DEPS + ["fe_kernels_gen.cuh"],
    "fe_tu_plane.cu": KERNEL_DEPS + ["fe_kernels_plane.cuh"],
    "fe_tu_line16.cu": KERNEL_DEPS + ["fe_kernels_plane.cuh", "fe_kernels_line.cuh", "fe_line_launch.inl"],
    "fe_tu_line8.cu": KERNEL_DEPS + ["fe_kernels_plane.cuh", "fe_kernels_line.cuh", "fe_line_launch.inl"],
    "fe_tu_oi.cu": KERNEL_DEPS + ["fe_kernels_oi.cuh"],
}

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "--fmad=true",
    "-Xcompiler", "-fPIC,-O2",
]

LIB_CHFSI = os.path.join(CSRC, "libfe_chfsi.so")
CHFSI_SOURCES = ["fe_chfsi.cu"]
CHFSI_DEPS = [os.path.join("..", "..", "include", "fe_chfsi.h"), FE_MF_H]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA library cannot be built (there is no CPU fallback)")


def _mtime(f: str) -> float:
    path = os.path.join(CSRC, f)
    return os.path.getmtime(path) if os.path.exists(path) else 0.0


def _obj(unit: str) -> str:
    return os.path.join(OBJ, unit[:-3] + ".o")


def _unit_stale(unit: str) -> bool:
    o = _obj(unit)
    if not os.path.exists(o):
        return True
    t = os.path.getmtime(o)
    return any(_mtime(f) > t for f in [unit] + UNITS[unit])


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(_mtime(f) > t for u in UNITS for f in [u] + UNITS[u])


def _stale(lib: str, files) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(_mtime(f) > t for f in files)


def build_chfsi(force: bool = False, verbose: bool = False) -> str:
    """libfe_chfsi.so; a separate library so that libfe_mf.so itself depends on nothing but the CUDA runtime."""
    build(force=False, verbose=verbose)
    if not force and not _stale(LIB_CHFSI, CHFSI_SOURCES + CHFSI_DEPS) and os.path.getmtime(LIB_CHFSI) >= os.path.getmtime(LIB):
        return LIB_CHFSI
    nvcc = nvcc_path()
    cuda_lib = os.path.join(os.path.dirname(os.path.dirname(os.path.realpath(nvcc))), "lib64")
    cmd = [nvcc] + NVCC_FLAGS + ["-shared"] + [os.path.join(CSRC, s) for s in CHFSI_SOURCES] + \
          ["-o", LIB_CHFSI, "-L" + CSRC, "-lfe_mf", "-lcublas", "-lcusolver",
           "-Xlinker", "-rpath=$ORIGIN", "-Xlinker", "-rpath=" + cuda_lib]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(" ".join(cmd) + "\n" + res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libfe_chfsi.so")
    return LIB_CHFSI


def _compile(unit: str, verbose: bool):
    cmd = [nvcc_path()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
          ["-c", os.path.join(CSRC, unit), "-o", _obj(unit)]
    res = subprocess.run(cmd, capture_output=True, text=True)
    return unit, cmd, res


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    todo = [u for u in UNITS if force or _unit_stale(u)]
    with ThreadPoolExecutor(max_workers=max(1, min(len(todo), os.cpu_count() or 1))) as pool:
        results = list(pool.map(lambda u: _compile(u, verbose), todo))
    failed = False
    for unit, cmd, res in results:
        if verbose or res.returncode != 0:
            sys.stderr.write(" ".join(cmd) + "\n" + res.stdout + res.stderr)
        failed = failed or res.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed building libfe_mf.so")
    cmd = [nvcc_path(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a"] + [_obj(u) for u in UNITS] + ["-o", LIB]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(" ".join(cmd) + "\n" + res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed linking libfe_mf.so")
    return LIB


PROBE_SRC = os.path.join(CSRC, "probe_pipes.cu")
PROBE_BIN = os.path.join(OBJ, "probe_pipes")


def build_probe(force: bool = False, verbose: bool = False) -> str:
    """The stand-alone box probe (DFMA vs DMMA, LDS vs DFMA; profiles/r2_probe_pipes.md): csrc/build/probe_pipes."""
    if not force and os.path.exists(PROBE_BIN) and os.path.getmtime(PROBE_BIN) >= os.path.getmtime(PROBE_SRC):
        return PROBE_BIN
    os.makedirs(OBJ, exist_ok=True)
    cmd = [nvcc_path(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-o", PROBE_BIN, PROBE_SRC]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(" ".join(cmd) + "\n" + res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building probe_pipes")
    return PROBE_BIN


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
    print(build_chfsi(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
    print(build_probe(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
