"""Parity of the SURVEY.md 8(f) NEXT-1 pieces (kappa at the quadrature points, GLL-lumped mass diagonal,
H~ = M^-1/2 (K + M^kappa) M^-1/2, Eq. B.1) with the CPU oracle, through the C-ABI binding."""
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
    """kind: 'uniform' (affine context), 'uniform_q' (uniform box, per-q-point context), 'perturbed_q'."""
    torch, orc, binding = env
    lo, hi = (0.0, -1.0, 0.5), (1.5, 0.5, 2.5)
    verts = None
    if kind == "perturbed_q":
        verts = inputs.perturbed_vertices(ncells, lo, hi, 0.15, 77)
    geom = binding.FE_GEOM_AFFINE if kind == "uniform" else binding.FE_GEOM_QPOINT
    op = binding.FeMf(ncells, p, sigma, bc, geom, lo, hi, verts)
    mesh = orc.Mesh(ncells, p, "periodic" if bc == inputs.BC_PERIODIC else "dirichlet", lo, hi, vertices=verts)
    return op, mesh


@pytest.mark.parametrize("p", [1, 2, 4, 6, 8])
@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_DIRICHLET])
@pytest.mark.parametrize("kind", ["uniform", "perturbed_q"])
def test_mass_diagonal(env, p, bc, kind):
    torch, orc, binding = env
    op, mesh = make_pair(env, p, bc, kind)
    M = op.mass_diagonal()
    Mo = orc.lumped_mass_diagonal(mesh)
    assert np.abs(M - Mo).max() <= 1e-14 * Mo.max()


@pytest.mark.parametrize("p", [2, 3, 5, 6, 7, 8])
@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_DIRICHLET])
@pytest.mark.parametrize("nvec", [8, 5])
def test_kappa_at_quadrature_points(env, p, bc, nvec):
    """K + M^kappa with an arbitrary kappa per quadrature point; nvec = 5 runs the fallback kernel."""
    torch, orc, binding = env
    op, mesh = make_pair(env, p, bc, "perturbed_q")
    ncell = 18
    kap = inputs.kappa_points(5 + p, ncell, (p + 1) ** 3)
    op.set_kappa(kap)
    X = inputs.multivector(31, mesh.ndof, nvec)
    Xd = torch.from_numpy(X).cuda()
    Yd = torch.full_like(Xd, float("nan"))
    op.apply(Xd, Yd, nvec)
    Yo = orc.Operator(mesh, 0.0, kappa=kap).apply(X)
    assert relerr(Yd.cpu().numpy(), Yo) <= TOL
    # back to the constant sigma
    op.set_kappa(None)
    op.apply(Xd, Yd, nvec)
    assert relerr(Yd.cpu().numpy(), orc.Operator(mesh, 0.7).apply(X)) <= TOL


def test_kappa_rejected_on_per_cell_metric_context(env):
    torch, orc, binding = env
    verts = inputs.uniform_vertices((3, 2, 3), (0, 0, 0), (1, 1, 1))
    op = binding.FeMf((3, 2, 3), 3, 1.0, inputs.BC_PERIODIC, binding.FE_GEOM_AFFINE, vertices=verts)
    with pytest.raises(binding.FeMfError) as e:
        op.set_kappa(np.zeros((18, 64)))
    assert e.value.code == binding.FE_MF_EINVAL


@pytest.mark.parametrize("p", [2, 6, 7])
@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_DIRICHLET])
def test_kappa_on_uniform_box_context(env, p, bc):
    """kappa without mass scaling on an affine (uniform box) context: served by the general kernel."""
    torch, orc, binding = env
    op, mesh = make_pair(env, p, bc, "uniform")
    kap = inputs.kappa_points(5 + p, 18, (p + 1) ** 3)
    op.set_kappa(kap)
    X = inputs.multivector(31, mesh.ndof, 8)
    Xd = torch.from_numpy(X).cuda()
    Yd = torch.full_like(Xd, float("nan"))
    op.apply(Xd, Yd, 8)
    assert relerr(Yd.cpu().numpy(), orc.Operator(mesh, 0.0, kappa=kap).apply(X)) <= TOL
    op.set_kappa(None)
    op.apply(Xd, Yd, 8)
    assert relerr(Yd.cpu().numpy(), orc.Operator(mesh, 0.7).apply(X)) <= TOL


def smooth_potential(orc, mesh):
    """Two Gaussian wells, a synthetic stand-in for the precomputed potential of PAPER.md:796."""
    xq = orc.quadrature_point_coordinates(mesh)
    c1, c2 = np.array([0.4, -0.5, 1.0]), np.array([1.1, 0.1, 2.0])
    return -8.0 * np.exp(-((xq - c1) ** 2).sum(-1) / 0.3) - 5.0 * np.exp(-((xq - c2) ** 2).sum(-1) / 0.5)


@pytest.mark.parametrize("p", [1, 2, 3, 4, 5, 6, 7, 8])
@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_DIRICHLET])
@pytest.mark.parametrize("kind", ["uniform", "uniform_k", "uniform_q", "perturbed_q"])
def test_mass_scaled_apply(env, p, bc, kind):
    """Y = M^-1/2 (K + M^kappa) M^-1/2 X.  'uniform' / 'uniform_k' (affine context, constant sigma /
    kappa per point) run on the Cartesian kernels with the mass-scaled tables, the others on the full-metric kernel."""
    torch, orc, binding = env
    op, mesh = make_pair(env, p, bc, "uniform" if kind == "uniform_k" else kind)
    kap = None
    if kind != "uniform":
        kap = smooth_potential(orc, mesh)
        op.set_kappa(kap)
    op.set_mass_scaling(True)
    oo = orc.Operator(mesh, 0.7, kappa=kap)
    d = 1.0 / np.sqrt(orc.lumped_mass_diagonal(mesh))
    for nvec in (8, 3, 16, 28):
        X = inputs.multivector(37, mesh.ndof, nvec)
        Xd = torch.from_numpy(X).cuda()
        Yd = torch.full_like(Xd, float("nan"))
        op.apply(Xd, Yd, nvec)
        assert relerr(Yd.cpu().numpy(), oo.apply_mass_scaled(X, d)) <= TOL, (nvec, op.kernel_name(nvec))
    # switching the scaling off restores H
    op.set_mass_scaling(False)
    op.apply(Xd, Yd, nvec)
    assert relerr(Yd.cpu().numpy(), oo.apply(X)) <= TOL


@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_DIRICHLET])
@pytest.mark.parametrize("kind,p", [("perturbed_q", 5), ("uniform", 6), ("uniform", 7), ("uniform", 3)])
def test_mass_scaled_axpby_eq_b1(env, bc, kind, p):
    """Y = a H~ X + b X + c Y (Eq. B.1)."""
    torch, orc, binding = env
    op, mesh = make_pair(env, p, bc, kind)
    kap = smooth_potential(orc, mesh)
    op.set_kappa(kap)
    op.set_mass_scaling(True)
    oo = orc.Operator(mesh, 0.0, kappa=kap)
    d = 1.0 / np.sqrt(orc.lumped_mass_diagonal(mesh))
    nvec = 12
    X = inputs.multivector(41, mesh.ndof, nvec)
    Y0 = inputs.multivector(43, mesh.ndof, nvec)
    a, b, c = 0.37, -1.25, 0.5
    Xd, Yd = torch.from_numpy(X).cuda(), torch.from_numpy(Y0).cuda()
    op.apply_axpby(a, Xd, c, b, Yd, nvec)
    expect = a * oo.apply_mass_scaled(X, d) + b * X + c * Y0      # constrained rows: H~ X = 0 there (reading 7)
    assert relerr(Yd.cpu().numpy(), expect) <= TOL


@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_DIRICHLET])
@pytest.mark.parametrize("p", [4, 6, 7, 8])
@pytest.mark.parametrize("kind", ["uniform", "uniform_q"])
def test_mass_scaled_chebyshev_filter(env, p, bc, kind):
    """Algorithm 6 lines 2-17 on H~ with mu = 1 and a smooth potential; on the affine context the
    one-launch-per-step recurrence of the Cartesian kernels (identity term added in the kernel)."""
    torch, orc, binding = env
    op, mesh = make_pair(env, p, bc, kind, ncells=(3, 3, 2))
    kap = smooth_potential(orc, mesh)
    op.set_kappa(kap)
    op.set_mass_scaling(True)
    oo = orc.Operator(mesh, 0.0, kappa=kap)
    d = 1.0 / np.sqrt(orc.lumped_mass_diagonal(mesh))
    nvec = 16
    X = inputs.multivector(47, mesh.ndof, nvec)
    app = lambda V: oo.apply_mass_scaled(V, d)
    b = orc.lanczos_upper_bound(app, X[:, 0].copy(), 12)
    a0 = -10.0
    a = a0 + 0.2 * (b - a0)
    m = 12
    Yo = orc.chebyshev_filter(app, X, m, a, b, a0)
    Xd = torch.from_numpy(X).cuda()
    Yd = torch.full_like(Xd, float("nan"))
    op.cheb_filter(Xd, Yd, nvec, m, a, b, a0)
    err = relerr(Yd.cpu().numpy(), Yo)
    assert err <= TOL, err
    if kind == "uniform":
        assert op.last_launch_count() <= m + 1


@pytest.mark.parametrize("kind", ["uniform", "perturbed_q"])
def test_host_path_with_mass_scaled_operator(env, kind):
    """fe_mf_apply_host (host buffers, column chunks on two streams) applies the operator the context is set to."""
    torch, orc, binding = env
    op, mesh = make_pair(env, 6, inputs.BC_PERIODIC, kind, ncells=(2, 2, 3))
    kap = smooth_potential(orc, mesh)
    op.set_kappa(kap)
    op.set_mass_scaling(True)
    oo = orc.Operator(mesh, 0.0, kappa=kap)
    d = 1.0 / np.sqrt(orc.lumped_mass_diagonal(mesh))
    nvec = 40                                       # three chunks, the last one partial
    X = inputs.multivector(61, mesh.ndof, nvec)
    Xh = torch.from_numpy(X).pin_memory(); Yh = torch.empty_like(Xh).pin_memory()
    op.apply_host(Xh, Yh, nvec)
    assert relerr(Yh.numpy(), oo.apply_mass_scaled(X, d)) <= TOL
