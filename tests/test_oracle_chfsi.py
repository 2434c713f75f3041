"""Pins of the oracle's Chebyshev filtered subspace iteration (Alg. 6)
against what the mathematics fixes: the converged Ritz values are eigenvalues (closed-form Laplacian spectrum, dense
eigendecomposition of the definition), one pass is a Rayleigh-Ritz on the filtered span.  No GPU."""
import numpy as np
import pytest

from oracle import fe_oracle as orc
from paper_2208_07129_b200 import inputs


def _problem(p=3, nc=3, L=2.0, kappa=None, bc="periodic"):
    mesh = orc.Mesh((nc,) * 3, p, bc, (0, 0, 0), (L,) * 3)
    op = orc.Operator(mesh, 0.0, ck=0.5, kappa=kappa)
    d = 1.0 / np.sqrt(orc.lumped_mass_diagonal(mesh))
    return mesh, (lambda V: op.apply_mass_scaled(V, d))


def test_chfsi_converges_to_laplacian_spectrum():
    """mu = 1/2, kappa = 1: lowest eigenvalues 1 + mu (2 pi/L)^2 {0, 1 x6, 2 x12} on the periodic cube."""
    L = 2.0
    mesh, app = _problem(p=4, nc=3, L=L, kappa=np.ones((27, 125)))
    U0 = inputs.multivector(7, mesh.ndof, 24)
    b = orc.lanczos_upper_bound(app, U0[:, 0].copy(), 12)
    U, lam, res, it = orc.chfsi_solve(app, U0, 19, 16, b, 0.3 * b, 0.0, 1e-8, 60)
    assert res[:19].max() <= 1e-8 and it < 60
    unit = 0.5 * (2 * np.pi / L) ** 2
    assert np.allclose(lam[:19], 1.0 + unit * np.array([0] + [1] * 6 + [2] * 12), rtol=2e-3)
    assert np.allclose(U.T @ U, np.eye(24), atol=1e-12)


def test_chfsi_matches_dense_eigendecomposition():
    """Dirichlet box with a potential well: the converged pairs are those of the dense matrix of the definition."""
    mesh = orc.Mesh((2, 3, 2), 3, "dirichlet", (0, 0, 0), (1.0, 1.5, 1.0))
    xq = orc.quadrature_point_coordinates(mesh)
    kap = -30.0 * np.exp(-((xq - np.array([0.4, 0.8, 0.5])) ** 2).sum(-1) / 0.1)
    op = orc.Operator(mesh, 0.0, ck=0.5, kappa=kap)
    d = 1.0 / np.sqrt(orc.lumped_mass_diagonal(mesh))
    app = lambda V: op.apply_mass_scaled(V, d)
    H = app(np.eye(mesh.ndof))
    nd = mesh.nd
    g = np.arange(mesh.ndof)
    ix, iy, iz = g % nd[0], (g // nd[0]) % nd[1], g // (nd[0] * nd[1])
    inner = ~((ix == 0) | (ix == nd[0] - 1) | (iy == 0) | (iy == nd[1] - 1) | (iz == 0) | (iz == nd[2] - 1))
    ref = np.linalg.eigvalsh(H[np.ix_(inner, inner)])
    U0 = inputs.multivector(9, mesh.ndof, 12)
    b = orc.lanczos_upper_bound(app, U0[:, 0].copy(), 12)
    U, lam, res, it = orc.chfsi_solve(app, U0, 8, 20, b, ref[0] + 0.2 * (b - ref[0]), ref[0] - 1.0, 1e-9, 80, free=inner)
    assert res[:8].max() <= 1e-9
    assert np.allclose(lam[:8], ref[:8], rtol=0, atol=1e-9 * abs(ref).max())
    assert np.abs(U[~inner]).max() == 0.0


def test_chfsi_one_pass_is_rayleigh_ritz_on_the_filtered_span():
    mesh, app = _problem(p=2, nc=3)
    U0 = inputs.multivector(11, mesh.ndof, 6)
    b = orc.lanczos_upper_bound(app, U0[:, 0].copy(), 10)
    U, lam, res = orc.chfsi_iterate(app, U0, 7, b, 0.4 * b, -0.1)
    Y = orc.chebyshev_filter(app, U0, 7, 0.4 * b, b, -0.1)
    # same span: projector onto span(Y) leaves U unchanged
    Qy, _ = np.linalg.qr(Y)
    assert np.allclose(Qy @ (Qy.T @ U), U, atol=1e-11)
    assert np.allclose(U.T @ U, np.eye(6), atol=1e-12)
    HU = app(U)
    assert np.allclose(U.T @ HU, np.diag(lam), atol=1e-10 * b)        # Ritz pairs: projected operator diagonal
    assert np.allclose(res, np.linalg.norm(HU - U * lam, axis=0), atol=1e-12 * b)
    assert np.all(np.diff(lam) >= 0)
