"""Pins of the second oracle (oracle/kron_oracle.py: the exactly integrated Kronecker closed form on uniform
Cartesian meshes) against what the mathematics fixes and against fe_oracle.Operator.apply, which
reaches the same operator from 3-D element matrices."""
import numpy as np
import pytest

from oracle import fe_oracle as orc
from oracle import kron_oracle as kro


def test_textbook_1d_matrices_p1_p2():
    """p = 1: M_e = h/6 [[2,1],[1,2]], K_e = 1/h [[1,-1],[-1,1]]; p = 2 (nodes -1, 0, 1):
    M_e = h/30 [[4,2,-1],[2,16,2],[-1,2,4]], K_e = 1/(3h) [[7,-8,1],[-8,16,-8],[1,-8,7]]."""
    h = 0.7
    M, K = kro.element_matrices_1d(1, h)
    assert np.allclose(M, h / 6 * np.array([[2, 1], [1, 2]]), rtol=0, atol=1e-15)
    assert np.allclose(K, 1 / h * np.array([[1, -1], [-1, 1]]), rtol=0, atol=1e-15)
    M, K = kro.element_matrices_1d(2, h)
    assert np.allclose(M, h / 30 * np.array([[4, 2, -1], [2, 16, 2], [-1, 2, 4]]), rtol=0, atol=1e-15)
    assert np.allclose(K, 1 / (3 * h) * np.array([[7, -8, 1], [-8, 16, -8], [1, -8, 7]]), rtol=0, atol=2e-14)


@pytest.mark.parametrize("p", [3, 4, 6, 7, 8])
def test_1d_matrices_invariants(p):
    """K 1 = 0 (constants have no gradient), 1^T M 1 = h, and the exact moments of x^k: sum_ij x_i^a M_ij x_j^b =
    int x^(a+b) on [-1,1] scaled, for a + b <= 2p (the basis reproduces monomials up to degree p)."""
    h = 1.3
    M, K = kro.element_matrices_1d(p, h)
    one = np.ones(p + 1)
    assert np.abs(K @ one).max() <= 1e-12 * np.abs(K).max()
    assert abs(one @ M @ one - h) <= 1e-14
    xi = np.asarray(orc.gll_nodes(p), dtype=np.float64)
    for a in range(p + 1):
        for b in range(p + 1):
            exact = (h / 2) * (0.0 if (a + b) % 2 else 2.0 / (a + b + 1))
            assert abs((xi ** a) @ M @ (xi ** b) - exact) <= 2e-14
            if a and b:   # int a x^(a-1) b x^(b-1) dxi * 2/h
                exact_k = (2 / h) * a * b * (0.0 if (a + b) % 2 else 2.0 / (a + b - 1))
                assert abs((xi ** a) @ K @ (xi ** b) - exact_k) <= 2e-12 * max(1.0, abs(exact_k))


@pytest.mark.parametrize("bc", ["periodic", "dirichlet"])
@pytest.mark.parametrize("p", [2, 3, 6, 7, 8])
def test_kronecker_apply_matches_cell_matrix_oracle(bc, p):
    """The two oracles agree element by element on anisotropic meshes (any transposed axis or wrong boundary row
    would show): relative max-norm 1e-13."""
    nc = (2, 3, 4) if p <= 3 else (2, 3, 2)
    lo, hi, sigma = (0.0, -1.0, 2.0), (1.0, 0.5, 4.4), 0.6
    mesh = orc.Mesh(nc, p, bc, lo, hi)
    rng = np.random.default_rng(100 + p)
    X = rng.uniform(-1, 1, (mesh.ndof, 3))
    Ya = orc.Operator(mesh, sigma).apply(X)
    Yb = kro.kronecker_apply(nc, p, bc, lo, hi, sigma, X)
    assert np.abs(Ya - Yb).max() <= 1e-13 * np.abs(Ya).max()
    if bc == "dirichlet":
        nd = mesh.nd
        Yb4 = Yb.reshape(nd[2], nd[1], nd[0], 3)
        assert np.all(Yb4[0] == 0) and np.all(Yb4[-1] == 0) and np.all(Yb4[:, 0] == 0) and np.all(Yb4[:, :, -1] == 0)


def test_exact_energy_of_a_separable_polynomial():
    """u = x^2 y - z^3 on [0,2]^3, natural mode replaced by a Dirichlet-free check on the periodic-free 1-D pieces:
    u^T A u for the separable terms equals the exact integrals (SURVEY.md 8(c) 'Exact energies': 312.888..., 64.6095...)."""
    p, nc, L = 3, 2, 2.0
    Me, Ke = kro.element_matrices_1d(p, L / nc)
    nd = nc * p + 1
    M1 = np.zeros((nd, nd)); K1 = np.zeros((nd, nd))
    for e in range(nc):
        idx = e * p + np.arange(p + 1)
        M1[np.ix_(idx, idx)] += Me; K1[np.ix_(idx, idx)] += Ke
    xi = np.asarray(orc.gll_nodes(p), dtype=np.float64)
    x = np.concatenate([[0.0]] + [(e + (xi[1:] + 1) / 2) * (L / nc) for e in range(nc)])
    X, Y, Z = np.meshgrid(x, x, x, indexing="ij")           # u[ix, iy, iz]
    u = X ** 2 * Y - Z ** 3
    def quad(Ax, Ay, Az):
        t = np.einsum("ia,abc->ibc", Ax, u); t = np.einsum("jb,ibc->ijc", Ay, t); t = np.einsum("kc,ijc->ijk", Az, t)
        return float((u * t).sum())
    grad2 = quad(K1, M1, M1) + quad(M1, K1, M1) + quad(M1, M1, K1)
    mass = quad(M1, M1, M1)
    # int_0^2 (2xy)^2 + x^4 + 9 z^4 and int (x^2 y - z^3)^2, closed forms
    e_grad = (4 * (8 / 3) * (8 / 3) * 2) + ((32 / 5) * 2 * 2) + (9 * (32 / 5) * 2 * 2)
    e_mass = (32 / 5) * (8 / 3) * 2 - 2 * (8 / 3) * 2 * 4 + (128 / 7) * 2 * 2
    assert abs(grad2 - e_grad) <= 1e-11 * e_grad and abs(e_grad - 312.8888888888889) < 1e-9
    assert abs(mass - e_mass) <= 1e-11 * e_mass and abs(e_mass - 64.60952380952381) < 1e-9
