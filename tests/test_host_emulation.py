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


# ---- the apply kernels that need neither TMA nor inline PTX, against the oracle -------------------------------------
import numpy as np  # noqa: E402

from oracle import dd_oracle as ddo  # noqa: E402
from oracle import fe_oracle as orc  # noqa: E402
from paper_2208_07129_b200 import inputs  # noqa: E402


def _emulator(tmp_path_factory, name, flags=()):
    """Compile tests/host/<name>.cpp against the shim; return run(kernel, ..., **options) -> Y [ndof][nvec].  Options
    (tests/host/emul_common.h): idw=float, layers="l0:l1", kappa=array, dscale=array."""
    tmp = tmp_path_factory.mktemp(name)
    exe = str(tmp / name)
    subprocess.run(["g++", "-std=c++20", "-O1", "-pthread", "-ffp-contract=off", "-Wno-unknown-pragmas", *flags, "-I", os.path.join(HOST, "shim"),
                    "-o", exe, os.path.join(HOST, name + ".cpp")], check=True)

    def run(kernel, p, nc, bc, zopen, geom_mode, nvec, sigma, lo, hi, X, verts=None, **options):
        xf, yf, vf = str(tmp / "x.bin"), str(tmp / "y.bin"), str(tmp / "v.bin")
        np.ascontiguousarray(X, dtype=np.float64).tofile(xf)
        cmd = [exe, kernel, str(p), *map(str, nc), str(bc), str(zopen), str(geom_mode), str(nvec), repr(float(sigma)),
               *[repr(float(v)) for v in lo], *[repr(float(v)) for v in hi], xf, yf]
        if verts is not None:
            np.ascontiguousarray(verts, dtype=np.float64).tofile(vf)
            cmd.append(vf)
        else:
            cmd.append("-")
        for key, val in options.items():
            if isinstance(val, np.ndarray):
                f = str(tmp / (key + ".bin"))
                np.ascontiguousarray(val, dtype=np.float64).tofile(f)
                cmd.append(f"{key}={f}")
            else:
                cmd.append(f"{key}={val}")
        res = subprocess.run(cmd, capture_output=True, text=True, timeout=600)
        assert res.returncode == 0, (res.returncode, res.stderr)
        return np.fromfile(yf, dtype=np.float64).reshape(-1, nvec)

    return run


@pytest.fixture(scope="module")
def emul_apply(tmp_path_factory):
    return _emulator(tmp_path_factory, "emul_apply")


@pytest.fixture(scope="module", params=["copies_at_issue", "copies_as_late_as_allowed"])
def emul_tma(tmp_path_factory, request):
    """Both legal extremes of the asynchronous bulk copies (tests/host/shim/cuda.h): at issue, and as late as the kernel's
    own waits allow (-DFE_EMUL_LAZY_TMA): a missing mbarrier wait or bulk-group wait makes the second one go wrong."""
    return _emulator(tmp_path_factory, "emul_tma", ["-DFE_EMUL_LAZY_TMA"] if request.param == "copies_as_late_as_allowed" else [])


def _relerr(a, b):
    return float(np.abs(a - b).max() / np.abs(b).max())


def _sheared_vertices(nc, lo, hi):
    """Vertices of an AFFINE image of the uniform grid (parallelepiped cells: J constant, full symmetric metric)."""
    g = [np.linspace(lo[d], hi[d], nc[d] + 1) for d in range(3)]
    Z, Yc, Xc = np.meshgrid(g[2], g[1], g[0], indexing="ij")
    A = np.array([[1.0, 0.25, -0.1], [0.05, 0.9, 0.2], [-0.15, 0.1, 1.1]])
    pts = np.stack([Xc, Yc, Z], axis=-1) @ A.T
    return pts                                                    # [(ncz+1)][(ncy+1)][(ncx+1)][3]


GENERAL_CASES = [
    # p, cells, bc, geometry, nvec
    (2, (2, 3, 2), "periodic", "box", 3),          # bv = 2: a vector tail
    (3, (2, 2, 3), "dirichlet", "box", 5),
    (2, (3, 2, 2), "periodic", "perturbed", 2),    # per-q-point metric (config 3's recipe)
    (3, (2, 2, 2), "dirichlet", "perturbed", 1),
    (2, (2, 2, 3), "dirichlet", "sheared", 4),     # per-cell constant, full symmetric metric
    (5, (2, 2, 2), "periodic", "box", 2),
]


@pytest.mark.parametrize("p,nc,bc,geometry,nvec", GENERAL_CASES)
def test_general_kernel_on_host_threads_matches_the_oracle(emul_apply, p, nc, bc, geometry, nvec):
    lo, hi, sigma = (0.0, -1.0, 0.5), (1.0, 0.5, 2.0), 0.7
    verts, mode = None, 0
    if geometry == "perturbed":
        verts, mode = inputs.perturbed_vertices(nc, lo, hi, 0.12, 77 + p), 2
    elif geometry == "sheared":
        verts, mode = _sheared_vertices(nc, lo, hi), 1
    mesh = orc.Mesh(nc, p, bc, lo, hi, vertices=verts)
    X = inputs.multivector(500 + p, mesh.ndof, nvec)
    Y = emul_apply("general", p, nc, 0 if bc == "periodic" else 1, 0, mode, nvec, sigma, lo, hi, X, verts)
    assert _relerr(Y, orc.Operator(mesh, sigma).apply(X)) <= 1e-12


CART_CASES = [
    # kernel, p, cells, bc, nvec
    ("cart", 2, (2, 3, 2), "periodic", 8),
    ("cart", 3, (2, 2, 3), "dirichlet", 11),       # a tail block of 3 vectors; even n: padded x-lines
    ("cart", 4, (3, 2, 2), "periodic", 5),
    ("cart", 5, (2, 2, 2), "dirichlet", 8),        # NT = TASKS / 2: two tasks per thread
    ("cart", 6, (2, 2, 2), "periodic", 9),
    ("cells", 3, (5, 2, 2), "periodic", 1),        # 8 cells of an x-row per block, ragged last group
    ("cells", 4, (5, 2, 2), "dirichlet", 2),
    ("cells", 6, (3, 2, 2), "periodic", 3),        # 2 cells x 3 vectors per block, 2 idle slots
]


@pytest.mark.parametrize("kernel,p,nc,bc,nvec", CART_CASES)
def test_even_odd_cartesian_kernel_on_host_threads_matches_the_oracle(emul_apply, kernel, p, nc, bc, nvec):
    """Also a check of the even-odd half tables of csrc/fe_eo_tables.h (Ns, Ns^T, Ds^T Ds / 2) end to end."""
    lo, hi, sigma = (0.0, 0.0, 0.0), (1.0, 1.5, 0.8), 0.6
    mesh = orc.Mesh(nc, p, bc, lo, hi)
    X = inputs.multivector(600 + p, mesh.ndof, nvec)
    Y = emul_apply(kernel, p, nc, 0 if bc == "periodic" else 1, 0, 0, nvec, sigma, lo, hi, X)
    assert _relerr(Y, orc.Operator(mesh, sigma).apply(X)) <= 1e-12


@pytest.mark.parametrize("kernel,nvec", [("general", 3), ("cart", 8), ("cells", 2)])
@pytest.mark.parametrize("bc", ["periodic", "dirichlet"])
def test_slab_flags_of_the_fallback_kernels_on_host_threads(emul_apply, kernel, nvec, bc):
    """NEXT-4: z_open bits (cut planes: no Dirichlet mask, no periodic wrap in z) in the kernels that mask through
    fe_z_masked, against the oracle's local operator of every task of a 3-slab decomposition."""
    p, nc, lo, hi, sigma = 3, (2, 2, 4), (0.0, 0.0, 0.0), (1.0, 1.0, 2.0), 0.9
    mesh = orc.Mesh(nc, p, bc, lo, hi)
    op = orc.Operator(mesh, sigma)
    X = inputs.multivector(700, mesh.ndof, nvec)
    hz = (hi[2] - lo[2]) / nc[2]
    layers = ddo.slab_layers(nc[2], 3)
    for t, (z0, z1) in enumerate(layers):
        rows, _ = ddo.slab_rows(mesh, z0, z1)
        U = X[rows].copy()
        zopen = 3 if bc == "periodic" else ((1 if t > 0 else 0) | (2 if t < len(layers) - 1 else 0))
        Y = emul_apply(kernel, p, (nc[0], nc[1], z1 - z0), 0 if bc == "periodic" else 1, zopen, 0, nvec, sigma,
                       (lo[0], lo[1], lo[2] + hz * z0), (hi[0], hi[1], lo[2] + hz * z1), U)
        assert _relerr(Y, ddo.slab_apply(op, z0, z1, U)) <= 1e-12, (t, zopen)


# ---- the persistent TMA kernels (plane, line, full metric) from their exact source ----------------------------------
# tests/host/shim/cuda.h: CUtensorMap as plain numbers (from the product's fe::tensor_map_desc), bulk tensor load with zero
# fill, bulk tensor reduce-add with clipping (aborts on a negative start coordinate or a misaligned tile, as the device
# faults), mbarrier phases with expected bytes, the dynamic item counter.

TMA_CASES = [
    # kernel, p, cells, bc, nvec, idw
    ("plane", 6, (2, 2, 2), "periodic", 16, 0.0),
    ("plane", 6, (2, 3, 2), "dirichlet", 32, 0.0),       # interior input map, trimmed output map, low-face zeroing
    ("plane", 6, (2, 2, 2), "periodic", 28, -0.7),       # vector tail of 12; identity term (the Chebyshev step's -c I)
    ("line16", 2, (3, 2, 2), "dirichlet", 20, 0.0),
    ("line16", 5, (2, 2, 2), "periodic", 16, 0.0),
    ("line16", 6, (2, 2, 2), "dirichlet", 16, 0.0),
    ("line8", 3, (2, 2, 3), "periodic", 6, 0.0),         # even n with 8-vector blocks: the pad node per x-row
    ("line8", 4, (2, 2, 2), "periodic", 8, 1.3),
    ("line8", 7, (2, 2, 2), "dirichlet", 8, 0.0),        # config 4's kernel
]


@pytest.mark.parametrize("kernel,p,nc,bc,nvec,idw", TMA_CASES)
def test_cartesian_tma_kernels_on_host_threads_match_the_oracle(emul_tma, kernel, p, nc, bc, nvec, idw):
    lo, hi, sigma = (0.0, 0.0, 0.0), (1.0, 1.5, 0.8), 0.6
    mesh = orc.Mesh(nc, p, bc, lo, hi)
    X = inputs.multivector(800 + p, mesh.ndof, nvec)
    Y = emul_tma(kernel, p, nc, 0 if bc == "periodic" else 1, 0, 0, nvec, sigma, lo, hi, X, idw=idw)
    assert _relerr(Y, orc.Operator(mesh, sigma).apply(X) + idw * X) <= 1e-12


GEN_CASES = [
    # p, cells, bc, geometry, nvec
    (2, (2, 3, 2), "periodic", "box", 4),                # a Cartesian mesh on the full-metric kernel (variant 7)
    (3, (2, 2, 3), "dirichlet", "box", 6),
    (2, (3, 2, 2), "periodic", "perturbed", 8),
    (3, (2, 2, 2), "dirichlet", "perturbed", 2),
    (5, (2, 2, 2), "periodic", "perturbed", 10),
    (3, (2, 2, 2), "periodic", "sheared", 4),            # one full symmetric metric per cell
    (8, (2, 2, 2), "periodic", "perturbed", 6),          # config 3's kernel: 4-vector blocks, 192 threads, a tail of 2
]


@pytest.mark.parametrize("p,nc,bc,geometry,nvec", GEN_CASES)
def test_full_metric_tma_kernel_on_host_threads_matches_the_oracle(emul_tma, p, nc, bc, geometry, nvec):
    lo, hi, sigma = (0.0, -1.0, 0.5), (1.0, 0.5, 2.0), 0.7
    verts, mode = None, 0
    if geometry == "perturbed":
        verts, mode = inputs.perturbed_vertices(nc, lo, hi, 0.12, 77 + p), 2
    elif geometry == "sheared":
        verts, mode = _sheared_vertices(nc, lo, hi), 1
    mesh = orc.Mesh(nc, p, bc, lo, hi, vertices=verts)
    X = inputs.multivector(500 + p, mesh.ndof, nvec)
    Y = emul_tma("gen", p, nc, 0 if bc == "periodic" else 1, 0, mode, nvec, sigma, lo, hi, X, verts)
    assert _relerr(Y, orc.Operator(mesh, sigma).apply(X)) <= 1e-12


@pytest.mark.parametrize("kernel,p,nvec", [("plane", 6, 16), ("line16", 5, 16), ("line8", 3, 8), ("gen", 3, 4)])
@pytest.mark.parametrize("bc", ["periodic", "dirichlet"])
def test_slab_flags_of_the_tma_kernels_on_host_threads(emul_tma, kernel, p, nvec, bc):
    """NEXT-4: the z_open bits in the tensor maps (per-direction trimming), the low-face zeroing, the wrap fix-ups:
    every task of a 3-slab decomposition against the oracle's local operator."""
    nc, lo, hi, sigma = (2, 2, 4), (0.0, 0.0, 0.0), (1.0, 1.0, 2.0), 0.9
    mesh = orc.Mesh(nc, p, bc, lo, hi)
    op = orc.Operator(mesh, sigma)
    X = inputs.multivector(700, mesh.ndof, nvec)
    hz = (hi[2] - lo[2]) / nc[2]
    layers = ddo.slab_layers(nc[2], 3)
    for t, (z0, z1) in enumerate(layers):
        rows, _ = ddo.slab_rows(mesh, z0, z1)
        U = X[rows].copy()
        zopen = 3 if bc == "periodic" else ((1 if t > 0 else 0) | (2 if t < len(layers) - 1 else 0))
        Y = emul_tma(kernel, p, (nc[0], nc[1], z1 - z0), 0 if bc == "periodic" else 1, zopen, 0, nvec, sigma,
                     (lo[0], lo[1], lo[2] + hz * z0), (hi[0], hi[1], lo[2] + hz * z1), U)
        assert _relerr(Y, ddo.slab_apply(op, z0, z1, U)) <= 1e-12, (t, zopen)


EIG_CASES = [
    # kernel, p, cells, bc, nvec, idw
    ("plane", 6, (2, 2, 2), "periodic", 16, 0.0),
    ("plane", 6, (2, 2, 3), "dirichlet", 16, 0.0),
    ("plane", 6, (2, 2, 2), "periodic", 16, -0.4),       # the filter step on H~: EIG + identity term
    ("line8", 4, (2, 3, 2), "periodic", 8, 0.0),
    ("line16", 5, (2, 2, 2), "dirichlet", 16, 0.0),
    ("line8", 7, (2, 2, 2), "periodic", 4, 0.9),
]


@pytest.mark.parametrize("kernel,p,nc,bc,nvec,idw", EIG_CASES)
def test_eigenproblem_operator_on_the_cartesian_tma_kernels_on_host_threads(emul_tma, kernel, p, nc, bc, nvec, idw):
    """NEXT-1: H~ = M^-1/2 (K + M^kappa) M^-1/2 on a uniform box: kappa per quadrature point, the mass
    scaling inside the interpolation tables (MAT_NSS of csrc/fe_eo_tables.h) and in the metric constants."""
    lo, hi = (0.0, 0.0, 0.0), (1.0, 1.5, 0.8)
    mesh = orc.Mesh(nc, p, bc, lo, hi)
    X = inputs.multivector(900 + p, mesh.ndof, nvec)
    kap = np.asarray(inputs.kappa_points(1234 + p, int(np.prod(nc)), (p + 1) ** 3))
    d = 1.0 / np.sqrt(orc.lumped_mass_diagonal(mesh))
    Y = emul_tma(kernel, p, nc, 0 if bc == "periodic" else 1, 0, 0, nvec, 0.0, lo, hi, X, kappa=kap, dscale=d, idw=idw)
    assert _relerr(Y, orc.Operator(mesh, 0.0, kappa=kap).apply_mass_scaled(X, d) + idw * X) <= 1e-12


@pytest.mark.parametrize("program,kernel,p,nc,bc,nvec", [("tma", "gen", 3, (2, 2, 2), "periodic", 4), ("tma", "gen", 2, (2, 3, 2), "dirichlet", 6),
                                                         ("apply", "general", 3, (2, 2, 2), "periodic", 3)])
def test_mass_scaled_operator_on_a_perturbed_mesh_on_host_threads(emul_tma, emul_apply, program, kernel, p, nc, bc, nvec):
    """d = diag(M)^-1/2 applied at extraction and assembly by the full-metric kernels."""
    lo, hi, sigma = (0.0, -1.0, 0.5), (1.0, 0.5, 2.0), 0.7
    verts = inputs.perturbed_vertices(nc, lo, hi, 0.12, 77 + p)
    mesh = orc.Mesh(nc, p, bc, lo, hi, vertices=verts)
    X = inputs.multivector(500 + p, mesh.ndof, nvec)
    d = 1.0 / np.sqrt(orc.lumped_mass_diagonal(mesh))
    run = emul_tma if program == "tma" else emul_apply
    Y = run(kernel, p, nc, 0 if bc == "periodic" else 1, 0, 2, nvec, sigma, lo, hi, X, verts, dscale=d)
    assert _relerr(Y, orc.Operator(mesh, sigma).apply_mass_scaled(X, d)) <= 1e-12


def test_kappa_on_a_uniform_box_on_the_general_kernel_on_host_threads(emul_apply):
    """kappa(x) without mass scaling runs on fe_apply_general (pick_kernel): the mass factor is det J * kappa_Q."""
    p, nc, lo, hi, nvec = 3, (2, 2, 2), (0.0, 0.0, 0.0), (1.0, 1.5, 0.8), 3
    mesh = orc.Mesh(nc, p, "periodic", lo, hi)
    X = inputs.multivector(960, mesh.ndof, nvec)
    kap = np.asarray(inputs.kappa_points(4321, int(np.prod(nc)), (p + 1) ** 3))
    Y = emul_apply("general", p, nc, 0, 0, 0, nvec, 0.0, lo, hi, X, kappa=kap)
    assert _relerr(Y, orc.Operator(mesh, 0.0, kappa=kap).apply(X)) <= 1e-12


@pytest.mark.parametrize("kernel,p,nc,bc,nvec", [("plane", 6, (2, 2, 4), "dirichlet", 16), ("line8", 3, (2, 2, 5), "periodic", 8),
                                                ("gen", 3, (2, 2, 4), "periodic", 4)])
def test_item_ranges_of_the_persistent_kernels_on_host_threads(emul_tma, kernel, p, nc, bc, nvec):
    """fe_mf_apply_host's z-slab pipeline launches the persistent kernels on a RANGE of cell layers (item0, item_count):
    the result is the sum of the contributions of exactly those cells (oracle: the same cells, one by one)."""
    lo, hi, sigma, l0, l1 = (0.0, 0.0, 0.0), (1.0, 1.5, 0.8), 0.6, 1, 3
    mesh = orc.Mesh(nc, p, bc, lo, hi)
    op = orc.Operator(mesh, sigma)
    X = inputs.multivector(950 + p, mesh.ndof, nvec)
    Y = emul_tma(kernel, p, nc, 0 if bc == "periodic" else 1, 0, 0, nvec, sigma, lo, hi, X, layers=f"{l0}:{l1}")
    Yo = np.zeros_like(X)
    for ez in range(l0, l1):
        for ey in range(nc[1]):
            for ex in range(nc[0]):
                idx, mask = mesh.cell_dofs(ex, ey, ez)
                U = X[idx].copy()
                if mask is not None:
                    U[mask] = 0.0
                W = op.cell_apply(ex, ey, ez, U)
                if mask is not None:
                    W[mask] = 0.0
                np.add.at(Yo, idx, W)
    assert _relerr(Y, Yo) <= 1e-12


# ---- n_q != n_p Gauss points per direction (NEXT-2) ------------------------------------------------------------------

@pytest.fixture(scope="module", params=["copies_at_issue", "copies_as_late_as_allowed"])
def emul_oi(tmp_path_factory, request):
    return _emulator(tmp_path_factory, "emul_oi", ["-DFE_EMUL_LAZY_TMA"] if request.param == "copies_as_late_as_allowed" else [])


OI_CASES = [
    # kernel, p, nq, cells, bc, geometry, nvec
    ("oi", 2, 5, (2, 3, 2), "periodic", "box", 4),
    ("oi", 3, 6, (2, 2, 2), "dirichlet", "perturbed", 6),
    ("oi", 4, 7, (2, 2, 2), "periodic", "perturbed", 5),        # odd nvec: a half-empty last block
    ("oi", 6, 9, (2, 2, 2), "periodic", "perturbed", 2),        # config 2's degree with the paper's n_q = n_p + 2
    ("oi_tma", 2, 5, (2, 3, 2), "periodic", "box", 4),          # the cell tile by bulk tensor copies; wrapped nodes by loads / atomics
    ("oi_tma", 3, 6, (2, 2, 2), "dirichlet", "perturbed", 6),   # boundary nodes zeroed in the tile
    ("oi_tma", 6, 9, (2, 2, 2), "periodic", "perturbed", 2),
    ("general_oi", 3, 5, (2, 2, 2), "periodic", "perturbed", 3),
    ("general_oi", 2, 7, (2, 2, 3), "dirichlet", "perturbed", 1),
    ("general_oi", 4, 7, (2, 2, 2), "periodic", "box", 1),      # n_q = n_p + 2 with one vector: the run-time kernel
]


@pytest.mark.parametrize("kernel,p,nq,nc,bc,geometry,nvec", OI_CASES)
def test_overintegration_kernels_on_host_threads_match_the_oracle(emul_oi, kernel, p, nq, nc, bc, geometry, nvec):
    """Rectangular tables from csrc/fe_oi_tables.h (N: n_q x n_p, the collocation derivative on the n_q points, their even /
    odd halves), per-point geometry at the n_q^3 points; fe_apply_oi in both of its modes."""
    lo, hi, sigma = (0.0, -1.0, 0.5), (1.0, 0.5, 2.0), 0.7
    verts, mode = None, 0
    if geometry == "perturbed":
        verts, mode = inputs.perturbed_vertices(nc, lo, hi, 0.12, 77 + p), 2
    mesh = orc.Mesh(nc, p, bc, lo, hi, vertices=verts)
    X = inputs.multivector(500 + p, mesh.ndof, nvec)
    Y = emul_oi(kernel, p, nc, 0 if bc == "periodic" else 1, 0, mode, nvec, sigma, lo, hi, X, verts, nq=nq)
    assert _relerr(Y, orc.Operator(mesh, sigma, nq=nq).apply(X)) <= 1e-12


def test_kappa_at_the_points_of_the_larger_rule_on_host_threads(emul_oi):
    p, nq, nc, nvec, lo, hi = 3, 6, (2, 2, 2), 4, (0.0, 0.0, 0.0), (1.0, 1.5, 0.8)
    mesh = orc.Mesh(nc, p, "periodic", lo, hi)
    X = inputs.multivector(77, mesh.ndof, nvec)
    kap = np.asarray(inputs.kappa_points(99, 8, nq ** 3))
    Y = emul_oi("oi", p, nc, 0, 0, 0, nvec, 0.0, lo, hi, X, nq=nq, kappa=kap)
    assert _relerr(Y, orc.Operator(mesh, 0.0, kappa=kap, nq=nq).apply(X)) <= 1e-12


def test_seeded_random_configurations_on_host_threads(emul_tma, emul_apply):
    """40 seeded random small configurations over all kernel families (degree, 1-3 cells per direction incl. one-cell-thick
    Dirichlet meshes, vector counts with and without tails, identity term): the oracle at 1e-12, and none of the aborts
    of the stand-ins (a reduction that starts at a negative coordinate, a misaligned tile)."""
    import random
    rnd = random.Random(20240807)
    lo, hi, sigma = (0.0, 0.0, 0.0), (1.0, 1.3, 0.7), 0.6
    degrees = {"plane": [6], "line16": [1, 2, 3, 5, 6], "line8": [1, 2, 3, 4, 7], "gen": [1, 2, 3, 5],
               "cart": [1, 2, 3, 4, 5, 6], "cells": [1, 2, 3, 4, 6], "general": [1, 2, 3, 4]}
    for case in range(40):
        kernel = rnd.choice(sorted(degrees))
        p = rnd.choice(degrees[kernel])
        bc = rnd.choice(["periodic", "dirichlet"])
        nc = tuple(rnd.randint(2 if bc == "periodic" else 1, 3) for _ in range(3))
        if bc == "dirichlet" and p == 1 and kernel in ("plane", "line16", "line8"):
            nc = tuple(max(c, 2) for c in nc)              # the trimmed maps need >= 3 nodes per direction (else pick_kernel takes kind 2)
        if kernel == "cells":
            nvec = rnd.choice([1, 2, 3])
        elif kernel in ("general", "cart"):
            nvec = rnd.choice([1, 2, 3, 5, 8, 9, 11])
        else:
            nvec = rnd.choice([2, 4, 6, 8, 10, 14, 16, 18, 20]) if p < 5 else rnd.choice([2, 6, 8, 12, 16])
        idw = rnd.uniform(-1, 1) if kernel in ("plane", "line16", "line8") and bc == "periodic" and rnd.random() < 0.3 else 0.0
        mesh = orc.Mesh(nc, p, bc, lo, hi)
        X = inputs.multivector(3000 + case, mesh.ndof, nvec)
        run = emul_tma if kernel in ("plane", "line16", "line8", "gen") else emul_apply
        Y = run(kernel, p, nc, 0 if bc == "periodic" else 1, 0, 0, nvec, sigma, lo, hi, X, **({"idw": idw} if idw else {}))
        Yo = orc.Operator(mesh, sigma).apply(X) + idw * X
        scale = np.abs(Yo).max()
        if scale == 0.0:                                   # every node on the Dirichlet boundary
            assert np.all(Y == 0.0), (case, kernel, p, nc, bc, nvec)
        else:
            assert np.abs(Y - Yo).max() <= 1e-12 * scale, (case, kernel, p, nc, bc, nvec, idw)


# ---- S9: the Chebyshev step as fe_cheb_filter composes it from accumulate launches ----------------------------------

@pytest.mark.parametrize("kernel,p,nc,bc,nvec,m", [("plane", 6, (2, 2, 2), "periodic", 16, 5), ("line8", 3, (2, 3, 2), "periodic", 8, 6),
                                                  ("line16", 5, (2, 2, 2), "dirichlet", 16, 4), ("plane", 6, (2, 2, 2), "dirichlet", 16, 3)])
def test_chebyshev_filter_from_accumulate_launches_on_host_threads(emul_tma, kernel, p, nc, bc, nvec, m):
    """The contract between fe_cheb_filter (csrc/fe_dispatch.cu) and the Cartesian TMA kernels, with the kernels run from
    their exact source: Alg. 6's recurrence in the scaled variables X_k = s_k U_k is a chain of accumulate launches
    U_{k-1} += al (A - c I) U_k, each ONE kernel launch with alpha = al and the identity term idw = -c al; on a Dirichlet
    mesh the kernels neither read nor write boundary rows, whose entries follow the scalar recurrence q_k and are written
    by the final scaling kernel.  The host recurrence below restates fe_cheb_filter's; the result is the oracle's filter."""
    lo, hi, sigma = (0.0, 0.0, 0.0), (1.0, 1.5, 0.8), 0.6
    mesh = orc.Mesh(nc, p, bc, lo, hi)
    op = orc.Operator(mesh, sigma)
    X0 = inputs.multivector(1700 + p, mesh.ndof, nvec)
    b = orc.lanczos_upper_bound(op.apply, inputs.uniform_pm1(1701, 0, mesh.ndof), 10)
    a, a0 = 0.35 * b, 0.0
    bcode = 0 if bc == "periodic" else 1

    def accumulate(al, W, Z):            # Z += al (A - c I) W in one launch
        return emul_tma(kernel, p, nc, bcode, 0, 0, nvec, sigma, lo, hi, W, alpha=repr(al), idw=repr(-c * al), z0=Z)

    e, c = (b - a) / 2.0, (b + a) / 2.0
    sig = e / (a0 - c)
    gamma = 2.0 / sig
    alpha1 = sig / e
    Uprev, Ucur = X0.copy(), accumulate(alpha1, X0, np.zeros_like(X0))
    s_prev = s_cur = 1.0
    q_prev, q_cur = 1.0, -c * alpha1
    for _ in range(2, m + 1):
        sig2 = 1.0 / (gamma - sig)
        alpha1, alpha2 = 2.0 * sig2 / e, -sig * sig2
        s_next = alpha2 * s_prev
        al = alpha1 * s_cur / s_next
        q_prev, q_cur = q_cur, -c * alpha1 * q_cur + alpha2 * q_prev
        Uprev, Ucur = Ucur, accumulate(al, Ucur, Uprev)
        s_prev, s_cur = s_cur, s_next
        sig = sig2
    Y = s_cur * Ucur
    if bc == "dirichlet":                # fe_scale2_kernel: boundary rows still hold x0 (or 0 in the buffer that started at 0)
        ix, iy, iz = np.meshgrid(*[np.arange(n) for n in mesh.nd], indexing="ij")
        bnd = (ix == 0) | (ix == mesh.nd[0] - 1) | (iy == 0) | (iy == mesh.nd[1] - 1) | (iz == 0) | (iz == mesh.nd[2] - 1)
        rows = (ix + mesh.nd[0] * (iy + mesh.nd[1] * iz))[bnd]
        Y[rows] = q_cur * X0[rows]
    Yo = orc.chebyshev_filter(op.apply, X0, m, a, b, a0)
    assert _relerr(Y, Yo) <= 1e-12
