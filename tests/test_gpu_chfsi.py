"""the Chebyshev filtered subspace iteration (Alg. 6) through
include/fe_chfsi.h against the oracle.  What is unique is compared (Ritz values, the Lanczos bound, converged
eigenvalues against the dense eigendecomposition of the definition); what is not (the basis inside a degenerate
eigenspace, signs) is checked for validity (orthonormality, residuals recomputed by the oracle)."""
import numpy as np
import pytest

from paper_2208_07129_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    from oracle import fe_oracle as orc
    from paper_2208_07129_b200 import binding, chfsi
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    chfsi.lib()
    return torch, orc, binding, chfsi


def setup(env, p, bc, ncells=(3, 2, 3), well=True):
    torch, orc, binding, chfsi = env
    lo, hi = (0.0, 0.0, 0.0), (1.5, 1.0, 1.5)
    op = binding.FeMf(ncells, p, 0.0, bc, binding.FE_GEOM_AFFINE, lo, hi)
    mesh = orc.Mesh(ncells, p, "periodic" if bc == inputs.BC_PERIODIC else "dirichlet", lo, hi)
    xq = orc.quadrature_point_coordinates(mesh)
    kap = 2.0 - 25.0 * np.exp(-((xq - np.array([0.6, 0.5, 0.8])) ** 2).sum(-1) / 0.15) if well else np.ones(xq.shape[:2])
    op.set_kappa(kap)
    op.set_mass_scaling(True)
    oo = orc.Operator(mesh, 0.0, kappa=kap)
    d = 1.0 / np.sqrt(orc.lumped_mass_diagonal(mesh))
    app = lambda V: oo.apply_mass_scaled(V, d)
    free = None
    if bc == inputs.BC_DIRICHLET:
        nd = mesh.nd
        g = np.arange(mesh.ndof)
        ix, iy, iz = g % nd[0], (g // nd[0]) % nd[1], g // (nd[0] * nd[1])
        free = ~((ix == 0) | (ix == nd[0] - 1) | (iy == 0) | (iy == nd[1] - 1) | (iz == 0) | (iz == nd[2] - 1))
    return op, mesh, app, free


@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_DIRICHLET])
def test_lanczos_bound(env, bc):
    torch, orc, binding, chfsi = env
    op, mesh, app, free = setup(env, 4, bc)
    v0 = inputs.uniform_pm1(91, 0, mesh.ndof)
    vo = v0.copy()
    if free is not None:
        vo[~free] = 0.0
    bo = orc.lanczos_upper_bound(app, vo, 10)
    h = chfsi.Chfsi(op, 4)
    b = h.lanczos_bound(torch.from_numpy(v0).cuda(), 10)
    assert abs(b - bo) <= 1e-10 * bo
    lam_max = np.linalg.eigvalsh(app(np.eye(mesh.ndof)))[-1]
    assert b >= lam_max


@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_DIRICHLET])
@pytest.mark.parametrize("p,nvec", [(3, 12), (6, 16)])
def test_one_pass_matches_oracle(env, p, nvec, bc):
    """Lines 2-20 once from the same block and bounds: same Ritz values; U orthonormal, in the filtered span, with
    the residuals the library reports."""
    torch, orc, binding, chfsi = env
    op, mesh, app, free = setup(env, p, bc, ncells=(2, 2, 3))
    U0 = inputs.multivector(93, mesh.ndof, nvec)
    b = orc.lanczos_upper_bound(app, U0[:, 0] * (1.0 if free is None else free), 10)
    lam_u, lam_min, m = 0.25 * b, -25.0, 9
    Uo, lam_o, res_o = orc.chfsi_iterate(app, U0 * (1.0 if free is None else free[:, None]), m, b, lam_u, lam_min, free)
    h = chfsi.Chfsi(op, nvec)
    Ud = torch.from_numpy(U0).cuda()
    lam, res = h.iterate(Ud, m, b, lam_u, lam_min)
    U = Ud.cpu().numpy()
    scale = np.abs(lam_o).max()
    assert np.abs(lam - lam_o).max() <= 1e-10 * scale
    assert np.abs(U.T @ U - np.eye(nvec)).max() <= 1e-12
    if free is not None:
        assert np.abs(U[~free]).max() == 0.0
    assert np.abs(np.linalg.norm(app(U) - U * lam, axis=0) - res).max() <= 1e-10 * scale
    assert np.abs(Uo @ (Uo.T @ U) - U).max() <= 1e-8              # same subspace
    t = h.last_timings()
    assert all(v >= 0 for v in t.values()) and t["filter"] > 0


@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_DIRICHLET])
def test_solve_converges_to_the_dense_spectrum(env, bc):
    torch, orc, binding, chfsi = env
    op, mesh, app, free = setup(env, 3, bc)
    H = app(np.eye(mesh.ndof))
    ref = np.linalg.eigvalsh(H if free is None else H[np.ix_(free, free)])
    nvec, nw = 16, 10
    U0 = inputs.multivector(95, mesh.ndof, nvec)
    h = chfsi.Chfsi(op, nvec)
    b = h.lanczos_bound(torch.from_numpy(U0[:, 0].copy()).cuda(), 12)
    Ud = torch.from_numpy(U0).cuda()
    tau = 1e-8
    lam, res, it = h.solve(Ud, nw, 20, b, ref[0] + 0.2 * (b - ref[0]), ref[0] - 1.0, tau, 80)
    assert it < 80 and res[:nw].max() <= tau
    assert np.abs(lam[:nw] - ref[:nw]).max() <= 1e-9 * np.abs(ref).max()
    U = Ud.cpu().numpy()
    assert np.abs(U.T @ U - np.eye(nvec)).max() <= 1e-12
    assert np.abs(np.linalg.norm(app(U) - U * lam, axis=0)[:nw]).max() <= 2 * tau
    # the oracle's own loop from the same start needs a comparable number of passes and finds the same values
    Uo, lam_o, res_o, it_o = orc.chfsi_solve(app, U0, nw, 20, b, ref[0] + 0.2 * (b - ref[0]), ref[0] - 1.0, tau, 80, free)
    assert abs(it - it_o) <= 1
    assert np.abs(lam[:nw] - lam_o[:nw]).max() <= 1e-9 * np.abs(ref).max()


def test_orthonormalize_and_rayleigh_ritz_entry_points(env):
    torch, orc, binding, chfsi = env
    op, mesh, app, free = setup(env, 4, inputs.BC_PERIODIC, ncells=(2, 2, 2))
    nvec = 8
    X = inputs.multivector(97, mesh.ndof, nvec)
    h = chfsi.Chfsi(op, nvec)
    Xd = torch.from_numpy(X).cuda()
    h.orthonormalize(Xd)
    Xo = Xd.cpu().numpy()
    assert np.abs(Xo.T @ Xo - np.eye(nvec)).max() <= 1e-13
    Q, _ = np.linalg.qr(X)
    assert np.abs(Q @ (Q.T @ Xo) - Xo).max() <= 1e-12               # same span
    Ud = torch.empty_like(Xd)
    lam, res = h.rayleigh_ritz(Xd, Ud)
    T = Xo.T @ app(Xo)
    assert np.abs(lam - np.linalg.eigvalsh((T + T.T) / 2)).max() <= 1e-11 * np.abs(lam).max()
    U = Ud.cpu().numpy()
    assert np.abs(np.linalg.norm(app(U) - U * lam, axis=0) - res).max() <= 1e-11 * np.abs(lam).max()
    # a rank-deficient block is refused
    X[:, 3] = X[:, 1]
    with pytest.raises(binding.FeMfError):
        h.orthonormalize(torch.from_numpy(X).cuda())


@pytest.mark.parametrize("nvec", [2, 5])
def test_small_and_odd_blocks(env, nvec):
    """Odd nvec (the operator falls back to its general kernel) and the smallest block the solve loop accepts."""
    torch, orc, binding, chfsi = env
    op, mesh, app, free = setup(env, 2, inputs.BC_DIRICHLET, ncells=(3, 3, 3))
    H = app(np.eye(mesh.ndof))
    ref = np.linalg.eigvalsh(H[np.ix_(free, free)])
    U0 = inputs.multivector(99, mesh.ndof, nvec)
    h = chfsi.Chfsi(op, nvec)
    b = h.lanczos_bound(torch.from_numpy(U0[:, 0].copy()).cuda(), 12)
    Ud = torch.from_numpy(U0).cuda()
    lam, res, it = h.solve(Ud, 1, 16, b, ref[0] + 0.3 * (b - ref[0]), ref[0] - 1.0, 1e-9, 200)
    assert res[0] <= 1e-9 and abs(lam[0] - ref[0]) <= 1e-9 * np.abs(ref).max()


def test_argument_errors(env):
    torch, orc, binding, chfsi = env
    op, mesh, app, free = setup(env, 2, inputs.BC_PERIODIC, ncells=(2, 2, 2))
    with pytest.raises(binding.FeMfError):
        chfsi.Chfsi(op, 0)
    h = chfsi.Chfsi(op, 4)
    U = torch.from_numpy(inputs.multivector(1, mesh.ndof, 4)).cuda()
    with pytest.raises(binding.FeMfError) as e:
        h.solve(U, 5, 8, 10.0, 5.0, 0.0, 1e-6)            # n_wanted > nvec
    assert e.value.code == binding.FE_MF_EINVAL
    with pytest.raises(binding.FeMfError) as e:
        h.iterate(U, 8, 10.0, 12.0, 0.0)                   # inverted filter interval: fe_cheb_filter refuses
    assert e.value.code == binding.FE_MF_EINVAL
    with pytest.raises(binding.FeMfError):
        h.rayleigh_ritz(U, U)
