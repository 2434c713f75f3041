"""Race check of the device code without a GPU: the host-thread builds of the kernels (tests/test_host_emulation.py,
tests/host/) compiled with ThreadSanitizer.  Every CUDA thread of a block is a real thread and shared memory is ordinary
memory, so a missing or misplaced __syncthreads() -- two threads of a block touching the same shared-memory word without
a barrier between them -- is a data race that TSan reports (checked: with the barrier between P2 and P3 of the plane
kernel removed it reports the race at the P3 tile read and the result is wrong).  Bulk tensor copies are executed by the
issuing thread AT ISSUE TIME, which is stricter than the device for a prefetch into a tile other threads might still
read, and blind to what only asynchrony can break (a missing wait on a bulk reduction that still reads its tile)."""
import os
import re
import subprocess

import numpy as np
import pytest

from oracle import fe_oracle as orc
from paper_2208_07129_b200 import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HOST = os.path.join(ROOT, "tests", "host")
CSRC = os.path.join(ROOT, "paper_2208_07129_b200", "csrc")
FLAGS = ["g++", "-std=c++20", "-O1", "-g", "-pthread", "-fsanitize=thread", "-ffp-contract=off", "-Wno-unknown-pragmas",
         "-I", os.path.join(HOST, "shim")]
ENV = dict(os.environ, TSAN_OPTIONS="halt_on_error=0 exitcode=66 report_signal_unsafe=0")


def tsan_works(tmp):
    """Some sandboxes forbid what TSan needs (personality / ASLR): skip rather than fail there."""
    src = os.path.join(tmp, "probe.cpp")
    open(src, "w").write("#include <thread>\nint x; int main() { std::thread a([]{ x = 1; }), b([]{ x = 2; }); a.join(); b.join(); return 0; }\n")
    exe = os.path.join(tmp, "probe")
    if subprocess.run(FLAGS[:1] + ["-std=c++20", "-O0", "-g", "-pthread", "-fsanitize=thread", "-o", exe, src], capture_output=True).returncode:
        return False
    r = subprocess.run([exe], capture_output=True, text=True, env=ENV)
    return "WARNING: ThreadSanitizer: data race" in r.stderr


@pytest.fixture(scope="module")
def tsan(tmp_path_factory):
    tmp = str(tmp_path_factory.mktemp("tsan"))
    if not tsan_works(tmp):
        pytest.skip("ThreadSanitizer cannot run in this environment")
    built = {}

    def program(name, extra_inc=()):
        if name not in built:
            exe = os.path.join(tmp, name)
            cmd = list(FLAGS)
            for inc in extra_inc:
                cmd += ["-I", inc]
            subprocess.run(cmd + ["-o", exe, os.path.join(HOST, name + ".cpp")], check=True)
            built[name] = exe
        return built[name]

    def run(name, args, extra_inc=()):
        r = subprocess.run([program(name, extra_inc)] + args, capture_output=True, text=True, env=ENV, timeout=1200)
        assert "ThreadSanitizer" not in r.stderr, r.stderr[:4000]
        assert r.returncode == 0, (r.returncode, r.stderr[:2000])
        return r

    return tmp, run


LO, HI, SIGMA = (0.0, 0.0, 0.0), (1.0, 1.5, 0.8), 0.6


def apply_args(tmp, kernel, p, nc, bc, nvec, geometry="box", **options):
    verts, mode = None, 0
    if geometry == "perturbed":
        verts, mode = inputs.perturbed_vertices(nc, LO, HI, 0.1, 31 + p), 2
    mesh = orc.Mesh(nc, p, bc, LO, HI, vertices=verts)
    X = inputs.multivector(5000 + p, mesh.ndof, nvec)
    xf, yf, vf = os.path.join(tmp, "x.bin"), os.path.join(tmp, "y.bin"), os.path.join(tmp, "v.bin")
    X.tofile(xf)
    args = [kernel, str(p), *map(str, nc), "0" if bc == "periodic" else "1", "0", str(mode), str(nvec), repr(SIGMA),
            *[repr(float(v)) for v in LO], *[repr(float(v)) for v in HI], xf, yf]
    if verts is not None:
        np.ascontiguousarray(verts).tofile(vf)
        args.append(vf)
    else:
        args.append("-")
    args += [f"{k}={v}" for k, v in options.items()]
    return args, (mesh, X, yf)


TMA = [("plane", 6, (2, 2, 2), "periodic", 16, "box", {"idw": -0.5}), ("plane", 6, (2, 2, 2), "dirichlet", 16, "box", {}),
       ("line16", 5, (2, 2, 2), "dirichlet", 16, "box", {}), ("line8", 3, (2, 2, 2), "periodic", 8, "box", {"idw": 0.5}),
       ("line8", 7, (2, 2, 2), "periodic", 8, "box", {}), ("gen", 3, (2, 2, 2), "periodic", 6, "perturbed", {}),
       ("gen", 3, (2, 2, 2), "dirichlet", 4, "perturbed", {}), ("gen", 8, (2, 2, 2), "periodic", 4, "perturbed", {})]


@pytest.mark.parametrize("kernel,p,nc,bc,nvec,geometry,options", TMA)
def test_tma_kernels_have_no_shared_memory_race(tsan, kernel, p, nc, bc, nvec, geometry, options):
    tmp, run = tsan
    args, (mesh, X, yf) = apply_args(tmp, kernel, p, nc, bc, nvec, geometry, **options)
    run("emul_tma", args)
    Y = np.fromfile(yf).reshape(-1, nvec)
    Yo = orc.Operator(mesh, SIGMA).apply(X) + options.get("idw", 0.0) * X
    assert np.abs(Y - Yo).max() <= 1e-12 * np.abs(Yo).max()


@pytest.mark.parametrize("program,kernel,p,nc,bc,nvec,geometry,options",
                         [("emul_apply", "general", 3, (2, 2, 2), "periodic", 3, "perturbed", {}), ("emul_apply", "cart", 4, (2, 2, 2), "dirichlet", 11, "box", {}),
                          ("emul_apply", "cells", 3, (3, 2, 2), "periodic", 2, "box", {}), ("emul_oi", "oi", 3, (2, 2, 2), "periodic", 4, "perturbed", {"nq": 6}),
                          ("emul_oi", "oi_tma", 3, (2, 2, 2), "periodic", 4, "perturbed", {"nq": 6}),
                          ("emul_oi", "general_oi", 2, (2, 2, 2), "dirichlet", 3, "perturbed", {"nq": 5})])
def test_fallback_and_overintegration_kernels_have_no_shared_memory_race(tsan, program, kernel, p, nc, bc, nvec, geometry, options):
    tmp, run = tsan
    args, _ = apply_args(tmp, kernel, p, nc, bc, nvec, geometry, **options)
    run(program, args)


def test_constraint_and_stream_kernels_have_no_race(tsan):
    tmp, run = tsan
    src = open(os.path.join(CSRC, "fe_constraints.cu")).read()
    m = re.search(r"// \[device-code-begin\][^\n]*\n(.*?)// \[device-code-end\]", src, flags=re.S)
    open(os.path.join(tmp, "emul_constraints_kernels.inc"), "w").write(m.group(1))
    run("emul_constraints", [], extra_inc=[tmp])
    run("emul_stream", [])
