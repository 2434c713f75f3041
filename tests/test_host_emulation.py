"""Device code run on the host (no GPU): the simple kernels of the library -- the two constraint kernels of
csrc/fe_constraints.cu and the streaming kernels of csrc/fe_kernels_stream.cuh (FP32 halo payload, axpby, scale, swap)
-- are compiled from their EXACT source with a small stand-in for the CUDA execution model (tests/host/shim/
cuda_runtime.h: one std::thread per CUDA thread, a std::barrier for __syncthreads, a lock for atomicAdd) and compared
with plain loops.  This checks the index arithmetic, grid-stride loops, tails and barrier placement of those kernels;
the GPU tests check the same kernels on the device."""
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HOST = os.path.join(ROOT, "tests", "host")
CSRC = os.path.join(ROOT, "paper_2208_07129_b200", "csrc")


def build_and_run(tmp, source, extra_inc=()):
    exe = os.path.join(tmp, os.path.splitext(os.path.basename(source))[0])
    cmd = ["g++", "-std=c++20", "-O1", "-pthread", "-ffp-contract=off", "-I", os.path.join(HOST, "shim")]
    for inc in extra_inc:
        cmd += ["-I", inc]
    subprocess.run(cmd + ["-o", exe, source], check=True)
    out = subprocess.run([exe], capture_output=True, text=True, check=True, timeout=600).stdout
    return [line.split() for line in out.splitlines()]


def test_constraint_kernels_on_host_threads(tmp_path):
    src = open(os.path.join(CSRC, "fe_constraints.cu")).read()
    m = re.search(r"// \[device-code-begin\][^\n]*\n(.*?)// \[device-code-end\]", src, flags=re.S)
    assert m, "markers missing in fe_constraints.cu"
    assert "fe_constraints_distribute_kernel" in m.group(1) and "fe_constraints_transpose_kernel" in m.group(1)
    (tmp_path / "emul_constraints_kernels.inc").write_text(m.group(1))
    rows = build_and_run(str(tmp_path), os.path.join(HOST, "emul_constraints.cpp"), extra_inc=[str(tmp_path)])
    assert len(rows) == 12                                     # 3 kernels-modes x 4 widths
    for name, nvec, err in rows:
        assert float(err) <= 1e-14, (name, nvec, err)


def test_stream_kernels_on_host_threads(tmp_path):
    rows = build_and_run(str(tmp_path), os.path.join(HOST, "emul_stream.cpp"))
    assert len(rows) == 8 * 5
    for name, count, bad in rows:
        assert int(bad) == 0, (name, count, bad)
