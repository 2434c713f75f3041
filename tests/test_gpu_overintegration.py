"""n_q = n_p + 2 Gauss points per direction (fe_mf_set_quadrature) against the oracle."""
import numpy as np
import pytest

from paper_2208_07129_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = 1e-12


@pytest.fixture(scope="module")
def env():
    import torch
    from oracle import fe_oracle as orc
    from paper_2208_07129_b200 import binding
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    binding.lib()
    return torch, orc, binding


def relerr(a, b):
    return float(np.abs(a - b).max() / np.abs(b).max())


def make_pair(env, p, bc, kind, ncells=(3, 2, 3), sigma=0.7):
    torch, orc, binding = env
    lo, hi = (0.0, -1.0, 0.5), (1.5, 0.5, 2.5)
    verts, geom = None, binding.FE_GEOM_AFFINE
    if kind == "perturbed_q":
        verts, geom = inputs.perturbed_vertices(ncells, lo, hi, 0.15, 77), binding.FE_GEOM_QPOINT
    elif kind == "sheared":
        verts = inputs.uniform_vertices(ncells, lo, hi) @ np.array([[1.0, 0.3, 0.1], [0.0, 1.1, 0.2], [0.0, 0.0, 0.9]]).T
    op = binding.FeMf(ncells, p, sigma, bc, geom, lo, hi, verts)
    mesh = orc.Mesh(ncells, p, "periodic" if bc == inputs.BC_PERIODIC else "dirichlet", lo, hi, vertices=verts)
    return op, mesh


def run(torch, op, X, nvec):
    Xd = torch.from_numpy(X).cuda()
    Yd = torch.full_like(Xd, float("nan"))
    op.apply(Xd, Yd, nvec)
    torch.cuda.synchronize()
    return Yd.cpu().numpy()


@pytest.mark.parametrize("p", [1, 2, 4, 6, 8])
@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_DIRICHLET])
@pytest.mark.parametrize("kind", ["uniform", "perturbed_q"])
def test_apply_with_np_plus_2_points(env, p, bc, kind):
    torch, orc, binding = env
    op, mesh = make_pair(env, p, bc, kind)
    nq = p + 3
    op.set_quadrature(nq)
    assert op.kernel_name(8) == "fe_apply_oi"
    oo = orc.Operator(mesh, 0.7, nq=nq)
    for nvec in (8, 3):
        X = inputs.multivector(51, mesh.ndof, nvec)
        assert relerr(run(torch, op, X, nvec), oo.apply(X)) <= TOL
    if kind == "perturbed_q":       # the two rules really differ on trilinear cells, and the default comes back
        base = orc.Operator(mesh, 0.7).apply(X)
        assert relerr(oo.apply(X), base) > 1e-9
        op.set_quadrature(p + 1)
        assert op.kernel_name(8) == "fe_apply_gen_tma"
        assert relerr(run(torch, op, X, 3), base) <= TOL


def test_sheared_cells_and_other_point_counts(env):
    torch, orc, binding = env
    op, mesh = make_pair(env, 3, inputs.BC_DIRICHLET, "sheared")
    X = inputs.multivector(53, mesh.ndof, 4)
    base = orc.Operator(mesh, 0.7).apply(X)
    for nq in (5, 6, 9):
        op.set_quadrature(nq)
        assert op.kernel_name(4) == ("fe_apply_oi" if nq == 6 else "fe_apply_general_oi")
        assert relerr(run(torch, op, X, 4), base) <= TOL       # affine cells: every rule with nq >= p + 1 is exact
    with pytest.raises(binding.FeMfError) as e:
        op.set_quadrature(3)
    assert e.value.code == binding.FE_MF_EINVAL
    with pytest.raises(binding.FeMfError):
        op.set_quadrature(13)


@pytest.mark.parametrize("kind", ["uniform", "perturbed_q"])
@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_DIRICHLET])
def test_kappa_mass_scaling_and_filter_with_np_plus_2_points(env, kind, bc):
    """kappa on the n_q^3 points, H~ = M^-1/2 (K + M^kappa) M^-1/2, Eq. B.1 and the Chebyshev filter on that rule."""
    torch, orc, binding = env
    p = 4
    op, mesh = make_pair(env, p, bc, kind)
    nq = p + 3
    op.set_quadrature(nq)
    xq = orc.quadrature_point_coordinates(mesh, nq)
    kap = -8.0 * np.exp(-((xq - np.array([0.4, -0.5, 1.0])) ** 2).sum(-1) / 0.3) + 1.0 + xq[..., 0]
    op.set_kappa(kap)
    oo = orc.Operator(mesh, 0.0, kappa=kap, nq=nq)
    nvec = 6
    X = inputs.multivector(55, mesh.ndof, nvec)
    assert relerr(run(torch, op, X, nvec), oo.apply(X)) <= TOL
    op.set_mass_scaling(True)
    d = 1.0 / np.sqrt(orc.lumped_mass_diagonal(mesh))
    app = lambda V: oo.apply_mass_scaled(V, d)
    assert relerr(run(torch, op, X, nvec), app(X)) <= TOL
    Z0 = inputs.multivector(57, mesh.ndof, nvec)
    Xd, Zd = torch.from_numpy(X).cuda(), torch.from_numpy(Z0).cuda()
    op.apply_axpby(0.4, Xd, -0.5, 1.5, Zd, nvec)
    assert relerr(Zd.cpu().numpy(), 0.4 * app(X) - 0.5 * Z0 + 1.5 * X) <= TOL
    b = orc.lanczos_upper_bound(app, X[:, 0].copy(), 12)
    Fo = orc.chebyshev_filter(app, X, 8, -10.0 + 0.2 * (b + 10.0), b, -10.0)
    Fd = torch.full_like(Xd, float("nan"))
    op.cheb_filter(Xd, Fd, nvec, 8, -10.0 + 0.2 * (b + 10.0), b, -10.0)
    err = relerr(Fd.cpu().numpy(), Fo)
    assert err <= TOL, err
    # dropping back to the default rule drops the kappa array (it belongs to the n_q^3 points)
    op.set_mass_scaling(False)
    op.set_quadrature(p + 1)
    assert relerr(run(torch, op, X, nvec), orc.Operator(mesh, 0.7).apply(X)) <= TOL


@pytest.mark.parametrize("p", [2, 5])
@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_DIRICHLET])
def test_interior_cells_take_the_tma_path(env, p, bc):
    """Every cell loads its tile with one bulk tensor copy and leaves through one bulk tensor reduction
    (fe_kernels_oi.cuh); cells that wrap around or touch the Dirichlet boundary patch the tile.  (4, 3, 4) cells have
    interior, wrap-around and boundary cells, and 6 vectors leave a vector tail for the TMA unit to zero-fill and clip."""
    torch, orc, binding = env
    op, mesh = make_pair(env, p, bc, "perturbed_q", ncells=(4, 3, 4))
    nq = p + 3
    op.set_quadrature(nq)
    oo = orc.Operator(mesh, 0.7, nq=nq)
    for nvec in (6, 2):
        assert op.kernel_name(nvec) == "fe_apply_oi"
        X = inputs.multivector(57, mesh.ndof, nvec)
        Y = run(torch, op, X, nvec)
        assert relerr(Y, oo.apply(X)) <= TOL
        op.set_variant(1)                     # the same kernel with loads and atomics on every cell
        Y1 = run(torch, op, X, nvec)
        op.set_variant(0)
        assert relerr(Y, Y1) <= 1e-14
    # Eq. B.1 through the TMA path: Z <- a A W + b Z + c W
    X = inputs.multivector(58, mesh.ndof, 4)
    Z = inputs.multivector(59, mesh.ndof, 4)
    Xd, Zd = torch.from_numpy(X).cuda(), torch.from_numpy(Z).cuda()
    op.apply_axpby(0.7, Xd, -0.3, 1.9, Zd, 4)
    torch.cuda.synchronize()
    assert relerr(Zd.cpu().numpy(), 0.7 * oo.apply(X) - 0.3 * Z + 1.9 * X) <= TOL
