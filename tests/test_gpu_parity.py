"""Parity of the CUDA path (through the C-ABI binding) with the CPU oracle, element by element on the
same seeded inputs.  Bar (BASELINE.json north_star): max|Y_gpu - Y_orc| / max|Y_orc| <= 1e-12."""
import numpy as np
import pytest

from paper_2208_07129_b200 import inputs

pytestmark = pytest.mark.gpu

TOL = 1e-12  # relative max-norm, north_star


@pytest.fixture(scope="module")
def env():
    import torch
    from oracle import fe_oracle as orc
    from paper_2208_07129_b200 import binding
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    binding.lib()
    return torch, orc, binding


def bc_name(bc):
    return "periodic" if bc == inputs.BC_PERIODIC else "dirichlet"


def oracle_mesh(orc, w):
    return orc.Mesh(w.ncells, w.p, bc_name(w.bc), w.box_lo, w.box_hi, vertices=inputs.workload_vertices(w))


def relerr(a, b):
    return float(np.abs(a - b).max() / np.abs(b).max())


def gpu_apply(torch, binding, w, X, nvec):
    op = binding.FeMf.from_workload(w)
    Xd = torch.from_numpy(X).cuda()
    Yd = torch.full_like(Xd, float("nan"))        # the apply must overwrite, not accumulate
    op.apply(Xd, Yd, nvec)
    torch.cuda.synchronize()
    assert op.last_launch_count() >= 1
    return Yd.cpu().numpy()


def check_apply(env, w, nvec=None):
    torch, orc, binding = env
    nvec = w.nvec if nvec is None else nvec
    X = inputs.multivector(w.seed, w.ndof, nvec)
    Y = gpu_apply(torch, binding, w, X, nvec)
    Yo = orc.Operator(oracle_mesh(orc, w), w.sigma).apply(X)
    err = relerr(Y, Yo)
    worst_col = max(relerr(Y[:, j:j + 1], Yo[:, j:j + 1]) for j in range(nvec))
    assert err <= TOL, (w.name, nvec, err, worst_col)
    return err


# ---------------------------------------------------------------- BASELINE.json configs at oracle-sized meshes
def test_cfg1_full(env):
    check_apply(env, inputs.configs()[1])


@pytest.mark.parametrize("nvec", [32, 5, 13])
def test_cfg2_scaled_dirichlet_p6(env, nvec):
    check_apply(env, inputs.configs()[2].scaled(4), nvec)


def test_cfg3_scaled_perturbed_p8(env):
    w = inputs.configs()[3].scaled(3)
    v = inputs.workload_vertices(w)
    assert np.abs(v - inputs.uniform_vertices(w.ncells, w.box_lo, w.box_hi)).max() > 0.05 / 16
    check_apply(env, w)


@pytest.mark.parametrize("nvec", [1, 8, 16, 32, 64])
def test_cfg4_scaled_p7_nvec_sweep(env, nvec):
    check_apply(env, inputs.configs()[4].scaled(3), nvec)


def test_cfg5_scaled_chebyshev(env):
    torch, orc, binding = env
    w = inputs.configs()[5].scaled(3, nvec=24)
    op_o = orc.Operator(oracle_mesh(orc, w), w.sigma)
    v0 = inputs.uniform_pm1(inputs.SEED_BASE + 5 + 200, 0, w.ndof)
    b = orc.lanczos_upper_bound(op_o.apply, v0, 10)
    assert b > w.cheb_a
    X = inputs.multivector(w.seed, w.ndof, w.nvec)
    Yo = orc.chebyshev_filter(op_o.apply, X, w.cheb_m, w.cheb_a, b, w.cheb_a0)
    op = binding.FeMf.from_workload(w)
    Xd = torch.from_numpy(X).cuda()
    Yd = torch.full_like(Xd, float("nan"))
    op.cheb_filter(Xd, Yd, w.nvec, w.cheb_m, w.cheb_a, b, w.cheb_a0)
    torch.cuda.synchronize()
    assert relerr(Yd.cpu().numpy(), Yo) <= TOL


# ---------------------------------------------------------------- every degree, both BCs, anisotropic mesh
@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_DIRICHLET])
@pytest.mark.parametrize("p", [1, 2, 3, 4, 5, 6, 7, 8])
def test_all_degrees_anisotropic(env, p, bc):
    w = inputs.Workload(f"aniso_p{p}", p, (2, 3, 4) if p <= 5 else (2, 3, 2), bc, inputs.GEOM_AFFINE, 0.7,
                        (0.0, -1.0, 2.0), (1.0, 0.5, 4.4), 6, 1000 + p)
    check_apply(env, w)


@pytest.mark.parametrize("p", [2, 5])
def test_per_qpoint_geometry_small_degrees(env, p):
    w = inputs.Workload(f"pert_p{p}", p, (3, 2, 4), inputs.BC_PERIODIC, inputs.GEOM_QPOINT, 1.3,
                        (0.0, 0.0, 0.0), (1.5, 1.0, 2.0), 7, 2000 + p, perturb=0.15)
    check_apply(env, w)


def test_per_qpoint_geometry_dirichlet(env):
    w = inputs.Workload("pert_dirichlet", 3, (3, 3, 3), inputs.BC_DIRICHLET, inputs.GEOM_QPOINT, 0.4,
                        (0.0, 0.0, 0.0), (1.0, 1.0, 1.0), 4, 2100, perturb=0.15)
    check_apply(env, w)


def test_affine_per_cell_sheared_mesh(env):
    """geom = AFFINE with explicit vertices: a sheared (parallelepiped) mesh, exact with one J per cell."""
    torch, orc, binding = env
    nc, p, sigma, nvec = (3, 2, 2), 4, 0.9, 8
    v = inputs.uniform_vertices(nc, (0, 0, 0), (1.0, 1.0, 1.0))
    S = np.array([[1.0, 0.3, 0.1], [0.0, 1.1, 0.2], [0.0, 0.0, 0.9]])
    v = v @ S.T
    mesh = orc.Mesh(nc, p, "dirichlet", vertices=v)
    X = inputs.multivector(77, mesh.ndof, nvec)
    Yo = orc.Operator(mesh, sigma).apply(X)
    op = binding.FeMf(nc, p, sigma, inputs.BC_DIRICHLET, inputs.GEOM_AFFINE, vertices=v)
    Xd = torch.from_numpy(X).cuda(); Yd = torch.empty_like(Xd)
    op.apply(Xd, Yd, nvec); torch.cuda.synchronize()
    assert relerr(Yd.cpu().numpy(), Yo) <= TOL


# ---------------------------------------------------------------- fused axpby, Chebyshev edge cases, host path
def test_apply_axpby(env):
    torch, orc, binding = env
    w = inputs.configs()[2].scaled(3, nvec=8)
    W = inputs.multivector(5, w.ndof, 8); Z = inputs.multivector(6, w.ndof, 8)
    AW = orc.Operator(oracle_mesh(orc, w), w.sigma).apply(W)
    op = binding.FeMf.from_workload(w)
    for alpha, beta, gamma in ((0.7, -0.3, 1.9), (2.0, 0.0, 0.5), (1.0, 1.0, 0.0), (-1.5, 0.0, 0.0)):
        Wd, Zd = torch.from_numpy(W).cuda(), torch.from_numpy(Z).cuda()
        op.apply_axpby(alpha, Wd, beta, gamma, Zd, 8); torch.cuda.synchronize()
        ref = alpha * AW + beta * Z + gamma * W
        assert relerr(Zd.cpu().numpy(), ref) <= TOL
        assert np.array_equal(Wd.cpu().numpy(), W)


@pytest.mark.parametrize("p,bc,nc,nvec", [(7, inputs.BC_PERIODIC, (2, 3, 2), 12), (7, inputs.BC_DIRICHLET, (3, 2, 2), 8),
                                          (6, inputs.BC_DIRICHLET, (2, 2, 4), 16), (4, inputs.BC_DIRICHLET, (3, 3, 3), 6),
                                          (5, inputs.BC_PERIODIC, (2, 2, 3), 20), (8, inputs.BC_DIRICHLET, (2, 2, 2), 4)])
@pytest.mark.parametrize("m", [1, 2, 7])
def test_chebyshev_scaled_recurrence_all_cartesian_kernels(env, m, p, bc, nc, nvec):
    """The one-launch-per-step filter on the line kernels (even and odd n, 8- and 16-vector blocks, pad-node tiles)
    and on Dirichlet meshes, where the boundary entries follow the scalar recurrence (closed form at the end)."""
    torch, orc, binding = env
    w = inputs.Workload("cheb_line", p, nc, bc, inputs.GEOM_AFFINE, 0.8, (0, 0, 0), (4.0, 6.0, 5.0), nvec, 500 + p)
    op_o = orc.Operator(oracle_mesh(orc, w), w.sigma)
    X = inputs.multivector(w.seed, w.ndof, w.nvec)
    a, b, a0 = 1.5, 12.0, -0.2
    Yo = orc.chebyshev_filter(op_o.apply, X, m, a, b, a0)
    Xprev = orc.chebyshev_filter(op_o.apply, X, m - 1, a, b, a0) if m > 1 else X
    op = binding.FeMf.from_workload(w)
    Xd = torch.from_numpy(X).cuda(); Yd = torch.full_like(Xd, float("nan"))
    op.cheb_filter(Xd, Yd, w.nvec, m, a, b, a0); torch.cuda.synchronize()
    assert relerr(Yd.cpu().numpy(), Yo) <= TOL
    assert relerr(Xd.cpu().numpy(), Xprev) <= TOL
    assert op.last_launch_count() <= m + 1


@pytest.mark.parametrize("nvec", [16, 28])
@pytest.mark.parametrize("m", [1, 2, 3, 8, 21])
def test_chebyshev_scaled_recurrence_plane_kernel(env, m, nvec):
    """p = 6, periodic (wrap in every direction), full and partial vector blocks: every filter step is one accumulate
    launch of the plane kernel, which adds the -c I part itself (partition-of-unity weights), in the scaled
    variables U_k = X_k / s_k."""
    torch, orc, binding = env
    w = inputs.Workload("cheb_plane", 6, (3, 2, 4), inputs.BC_PERIODIC, inputs.GEOM_AFFINE, 1.0, (0, 0, 0), (7.5, 5.0, 10.0),
                        nvec, 77)
    op_o = orc.Operator(oracle_mesh(orc, w), w.sigma)
    X = inputs.multivector(w.seed, w.ndof, w.nvec)
    a, b, a0 = 1.0, 3.0, -0.05
    Yo = orc.chebyshev_filter(op_o.apply, X, m, a, b, a0)
    Xprev = orc.chebyshev_filter(op_o.apply, X, m - 1, a, b, a0) if m > 1 else X
    op = binding.FeMf.from_workload(w)
    Xd = torch.from_numpy(X).cuda(); Yd = torch.full_like(Xd, float("nan"))
    op.cheb_filter(Xd, Yd, w.nvec, m, a, b, a0); torch.cuda.synchronize()
    assert relerr(Yd.cpu().numpy(), Yo) <= TOL
    assert relerr(Xd.cpu().numpy(), Xprev) <= TOL           # X holds iterate m-1 (header contract)
    assert op.last_launch_count() <= m + 1                  # m accumulate launches + one final scaling


@pytest.mark.parametrize("m", [1, 2, 3, 6])
def test_chebyshev_small_degrees_and_x_scratch(env, m):
    torch, orc, binding = env
    w = inputs.Workload("cheb", 3, (3, 3, 3), inputs.BC_DIRICHLET, inputs.GEOM_AFFINE, 1.0, (0, 0, 0), (3.0, 3.0, 3.0),
                        5, 31)
    op_o = orc.Operator(oracle_mesh(orc, w), w.sigma)
    X = inputs.multivector(w.seed, w.ndof, w.nvec)
    a, b, a0 = 1.0, 9.0, -0.1
    Yo = orc.chebyshev_filter(op_o.apply, X, m, a, b, a0)
    Xprev = orc.chebyshev_filter(op_o.apply, X, m - 1, a, b, a0) if m > 1 else X
    op = binding.FeMf.from_workload(w)
    Xd = torch.from_numpy(X).cuda(); Yd = torch.empty_like(Xd)
    op.cheb_filter(Xd, Yd, w.nvec, m, a, b, a0); torch.cuda.synchronize()
    assert relerr(Yd.cpu().numpy(), Yo) <= TOL
    assert relerr(Xd.cpu().numpy(), Xprev) <= TOL           # X holds iterate m-1 (header contract)


@pytest.mark.parametrize("nvec", [1, 2, 3])
@pytest.mark.parametrize("p,bc,nc", [(7, inputs.BC_PERIODIC, (5, 2, 2)), (6, inputs.BC_DIRICHLET, (9, 2, 3)),
                                     (4, inputs.BC_PERIODIC, (3, 3, 2)), (2, inputs.BC_DIRICHLET, (11, 2, 2))])
def test_few_vectors_cells_as_slots(env, p, bc, nc, nvec):
    """1-3 vectors on a Cartesian mesh: the tile slots hold several cells of an x-row (ragged last group of cells)."""
    w = inputs.Workload(f"few_p{p}", p, nc, bc, inputs.GEOM_AFFINE, 0.6, (0.0, 0.0, 0.0), (2.5, 1.0, 1.5), nvec, 900 + p)
    check_apply(env, w)


def test_cuda_graph_capture(env):
    """The entry points only enqueue work on the caller's stream (no host synchronisation, no allocation after the
    first call): an apply and a filter can be captured in a CUDA graph and replayed (config 1 is launch-bound)."""
    torch, orc, binding = env
    w = inputs.configs()[1]
    X = inputs.multivector(w.seed, w.ndof, w.nvec)
    oo = orc.Operator(oracle_mesh(orc, w), w.sigma)
    Yo = oo.apply(X)
    Fo = orc.chebyshev_filter(oo.apply, X, 4, 50.0, 400.0, 0.0)
    op = binding.FeMf.from_workload(w)
    Xd = torch.from_numpy(X).cuda(); Yd = torch.empty_like(Xd); Xf = Xd.clone(); Yf = torch.empty_like(Xd)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        op.apply(Xd, Yd, w.nvec, stream=s); op.cheb_filter(Xf, Yf, w.nvec, 4, 50.0, 400.0, 0.0, stream=s)   # warm-up (function attributes)
        s.synchronize()
        g = torch.cuda.CUDAGraph()
        Xf.copy_(Xd)
        with torch.cuda.graph(g, stream=s):
            op.apply(Xd, Yd, w.nvec, stream=s)
            op.cheb_filter(Xf, Yf, w.nvec, 4, 50.0, 400.0, 0.0, stream=s)
        Yd.fill_(float("nan")); Yf.fill_(float("nan")); Xf.copy_(Xd)
        g.replay()
        s.synchronize()
    assert relerr(Yd.cpu().numpy(), Yo) <= TOL
    assert relerr(Yf.cpu().numpy(), Fo) <= TOL


def test_apply_host_path(env):
    torch, orc, binding = env
    for nvec in (3, 32):
        w = inputs.configs()[2].scaled(3, nvec=nvec)
        X = inputs.multivector(w.seed, w.ndof, nvec)
        Yo = orc.Operator(oracle_mesh(orc, w), w.sigma).apply(X)
        op = binding.FeMf.from_workload(w)
        Xh = torch.from_numpy(X).pin_memory(); Yh = torch.empty_like(Xh).pin_memory()
        op.apply_host(Xh, Yh, nvec)
        assert relerr(Yh.numpy(), Yo) <= TOL


def test_fill_uniform_bit_exact(env):
    torch, orc, binding = env
    out = torch.empty(100003, dtype=torch.float64, device="cuda")
    binding.fill_uniform(out, inputs.SEED_BASE + 2, offset=12345); torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), inputs.uniform_pm1(inputs.SEED_BASE + 2, 12345, 100003))


def test_error_codes(env):
    torch, orc, binding = env
    F = binding.FeMf
    with pytest.raises(binding.FeMfError) as e:
        F((2, 2, 2), 9, 1.0, 0)
    assert e.value.code == binding.FE_MF_EINVAL
    with pytest.raises(binding.FeMfError):
        F((1, 2, 2), 2, 1.0, inputs.BC_PERIODIC)               # periodic cell neighbouring itself
    with pytest.raises(binding.FeMfError):
        F((2, 2, 2), 2, 1.0, 0, box_lo=(0, 0, 0), box_hi=(1, 0, 1))
    v = inputs.uniform_vertices((2, 2, 2), (0, 0, 0), (1, 1, 1)); v[1, 1, 1] = [5.0, 5.0, 5.0]   # inverted cell
    with pytest.raises(binding.FeMfError):
        F((2, 2, 2), 2, 1.0, inputs.BC_DIRICHLET, inputs.GEOM_QPOINT, vertices=v)
    op = F((2, 2, 2), 2, 1.0, inputs.BC_PERIODIC)
    X = torch.zeros(op.ndofs * 2, dtype=torch.float64, device="cuda"); Y = torch.zeros_like(X)
    with pytest.raises(binding.FeMfError):
        op.apply(X, X, 2)                                        # aliasing
    with pytest.raises(binding.FeMfError) as e:
        op.cheb_filter(X, Y, 2, 5, 2.0, 1.0, 0.0)                # inverted interval (reading 12)
    assert e.value.code == binding.FE_MF_EINVAL
    with pytest.raises(binding.FeMfError):
        op.cheb_filter(X, Y, 2, 0, 1.0, 2.0, 0.0)
    with pytest.raises(binding.FeMfError):
        op.cheb_filter(X, Y, 2, 3, 1.0, 2.0, 1.5)                # a0 >= a


def test_unit_cube_config5_interval_is_rejected(env):
    """DESIGN.md reading 12: on the unit cube lambda_max(K+M) < 2.0 at p=6, h=1/16, so [2.0, b] is inverted."""
    torch, orc, binding = env
    op = binding.FeMf((4, 4, 4), 6, 1.0, inputs.BC_PERIODIC, box_hi=(0.25, 0.25, 0.25))
    X = torch.zeros(op.ndofs, dtype=torch.float64, device="cuda"); Y = torch.zeros_like(X)
    with pytest.raises(binding.FeMfError):
        op.cheb_filter(X, Y, 1, 20, 2.0, 0.3, 0.0)


@pytest.mark.parametrize("variant", [1, 2, 8, 10, 11])
@pytest.mark.parametrize("p,bc", [(6, inputs.BC_DIRICHLET), (7, inputs.BC_PERIODIC), (8, inputs.BC_PERIODIC), (4, inputs.BC_PERIODIC)])
def test_kernel_variants(env, variant, p, bc):
    """variant 1 = general fallback kernel, 2 = even-odd Cartesian kernel with one vector per thread (LDG/RED),
    8 = plane kernel (p = 6 only; other degrees keep their default), 10 / 11 = line kernel with 16 / 8 vectors per block."""
    torch, orc, binding = env
    w = inputs.Workload(f"var_p{p}", p, (3, 2, 3), bc, inputs.GEOM_AFFINE, 0.8, (0.0, 0.0, 0.0), (1.5, 1.0, 2.0), 20, 500 + p)
    X = inputs.multivector(w.seed, w.ndof, w.nvec)
    Yo = orc.Operator(oracle_mesh(orc, w), w.sigma).apply(X)
    op = binding.FeMf.from_workload(w)
    op.set_variant(variant)
    Xd = torch.from_numpy(X).cuda(); Yd = torch.empty_like(Xd)
    op.apply(Xd, Yd, w.nvec); torch.cuda.synchronize()
    assert relerr(Yd.cpu().numpy(), Yo) <= TOL


@pytest.mark.parametrize("variant", [0, 8])
@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_DIRICHLET])
def test_plane_kernel_many_layers(env, bc, variant):
    """p = 6, 9 cell layers in z, 40 vectors (a partial last block of 8: the default is then the line kernel, variant 8
    forces the plane kernel): plain apply and Z <- beta Z + gamma W + alpha A W."""
    torch, orc, binding = env
    w = inputs.Workload("plane_layers", 6, (2, 3, 9), bc, inputs.GEOM_AFFINE, 0.7, (0.0, 0.0, 0.0), (1.0, 1.5, 3.0), 40, 4242)
    X = inputs.multivector(w.seed, w.ndof, w.nvec)
    Z0 = inputs.multivector(w.seed + 1, w.ndof, w.nvec)
    Yo = orc.Operator(oracle_mesh(orc, w), w.sigma).apply(X)
    op = binding.FeMf.from_workload(w); op.set_variant(variant)
    assert op.kernel_name(w.nvec) == ("fe_apply_cart_plane" if variant == 8 else "fe_apply_cart_line")
    Xd = torch.from_numpy(X).cuda(); Yd = torch.full_like(Xd, float("nan"))
    op.apply(Xd, Yd, w.nvec); torch.cuda.synchronize()
    assert relerr(Yd.cpu().numpy(), Yo) <= TOL
    assert op.last_launch_count() == 1                      # the zero fill is a driver memset
    Zd = torch.from_numpy(Z0).cuda()
    op.apply_axpby(0.3, Xd, 0.5, -0.25, Zd, w.nvec); torch.cuda.synchronize()
    assert relerr(Zd.cpu().numpy(), 0.5 * Z0 - 0.25 * X + 0.3 * Yo) <= TOL
    assert op.last_launch_count() == 2
    Zd = torch.from_numpy(Z0).cuda()
    op.apply_axpby(0.3, Xd, 0.0, -0.25, Zd, w.nvec); torch.cuda.synchronize()
    assert relerr(Zd.cpu().numpy(), -0.25 * X + 0.3 * Yo) <= TOL


@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_DIRICHLET])
@pytest.mark.parametrize("p", [1, 2, 3, 4, 5, 6, 7, 8])
def test_general_metric_tma_kernel_all_degrees(env, p, bc):
    """Per-q-point geometry, even nvec: the persistent TMA kernel for a full symmetric metric (with vector tail)."""
    nc = (3, 2, 3) if p <= 6 else (2, 2, 3)
    w = inputs.Workload(f"gen_p{p}", p, nc, bc, inputs.GEOM_QPOINT, 0.9, (0.0, 0.0, 0.0), (1.5, 1.0, 2.0), 10, 3000 + p,
                        perturb=0.15)
    check_apply(env, w)


@pytest.mark.parametrize("p", [3, 6, 8])
def test_general_metric_kernel_on_uniform_mesh(env, p):
    """variant 7 forces the full-metric kernel on a Cartesian mesh (metric read from memory, off-diagonals 0)."""
    torch, orc, binding = env
    w = inputs.Workload(f"gen_uniform_p{p}", p, (3, 2, 2), inputs.BC_PERIODIC, inputs.GEOM_AFFINE, 1.2, (0, 0, 0), (1.5, 1.0, 1.0), 8, 3100 + p)
    X = inputs.multivector(w.seed, w.ndof, w.nvec)
    Yo = orc.Operator(oracle_mesh(orc, w), w.sigma).apply(X)
    op = binding.FeMf.from_workload(w); op.set_variant(7)
    Xd = torch.from_numpy(X).cuda(); Yd = torch.empty_like(Xd)
    op.apply_axpby(0.5, Xd, 0.0, 0.0, Yd, w.nvec); torch.cuda.synchronize()
    assert relerr(Yd.cpu().numpy(), 0.5 * Yo) <= TOL
