"""Pins of the oracle's NEXT-1 pieces: the GLL-lumped mass diagonal, the weighted mass matrix
M^kappa with kappa given at the quadrature points, and H~ = M^-1/2 (K + M^kappa) M^-1/2 (Eq. B.1).
No GPU, no CUDA path."""
from fractions import Fraction

import numpy as np
import pytest

from oracle import fe_oracle as orc
from paper_2208_07129_b200 import inputs


# ------------------------------------------------------------------ GLL weights
def test_gll_weights_textbook_values():
    """Printed values of the Lobatto rule (any quadrature table): p = 1..4."""
    table = {1: [1, 1], 2: [Fraction(1, 3), Fraction(4, 3), Fraction(1, 3)],
             3: [Fraction(1, 6), Fraction(5, 6), Fraction(5, 6), Fraction(1, 6)],
             4: [Fraction(1, 10), Fraction(49, 90), Fraction(32, 45), Fraction(49, 90), Fraction(1, 10)]}
    for p, w in table.items():
        assert np.allclose(orc.gll_weights(p).astype(float), [float(v) for v in w], atol=2e-16, rtol=0)


@pytest.mark.parametrize("p", [1, 2, 3, 4, 5, 6, 7, 8])
def test_gll_weights_exactness(p):
    """The (p+1)-point Lobatto rule integrates degree <= 2p-1 exactly and degree 2p with a negative error."""
    x, w = orc.gll_nodes(p).astype(float), orc.gll_weights(p).astype(float)
    for k in range(0, 2 * p):
        exact = 2.0 / (k + 1) if k % 2 == 0 else 0.0
        assert abs((w * x ** k).sum() - exact) < 4e-15
    assert (w * x ** (2 * p)).sum() > 2.0 / (2 * p + 1) + 1e-6 * 0.5 ** p


# ------------------------------------------------------------------ lumped mass
def _perturbed_mesh(p, bc, ncells=(2, 3, 2), lo=(0.0, -1.0, 0.5), hi=(1.5, 1.0, 2.0)):
    v = inputs.perturbed_vertices(ncells, lo, hi, 0.15, 7) if bc != "periodic" else None
    return orc.Mesh(ncells, p, bc, lo, hi, vertices=v)


@pytest.mark.parametrize("p", [2, 3, 5])
def test_lumped_mass_total_is_volume(p):
    """sum_i M_ii = |Omega|: det J of a trilinear cell has degree <= 2 per direction, the rule is exact to 2p-1."""
    m = _perturbed_mesh(p, "natural")
    M = orc.lumped_mass_diagonal(m)
    assert M.min() > 0
    assert abs(M.sum() - 1.5 * 2.0 * 1.5) < 1e-13


@pytest.mark.parametrize("p,perturbed", [(1, False), (2, False), (3, True), (4, True), (6, True)])
def test_lumped_mass_is_row_sum_of_consistent_mass(p, perturbed):
    """M_ii(lumped) = int N_i = sum_j M_ij whenever the Lobatto rule integrates N_i det J exactly
    (degree p + 2 <= 2p - 1 on trilinear cells, degree p on affine ones)."""
    if perturbed:
        m = _perturbed_mesh(p, "natural", ncells=(2, 2, 1))
    else:
        m = orc.Mesh((2, 1, 3), p, "natural", (0, 0, 0), (1.0, 2.0, 0.5))
    consistent = orc.Operator(m, 1.0, ck=0.0, cm=1.0)
    rows = consistent.apply(np.ones(m.ndof))
    assert np.allclose(orc.lumped_mass_diagonal(m), rows, rtol=0, atol=1e-14 * rows.max() * 10)


def test_lumped_mass_periodic_uniform_closed_form():
    """Uniform periodic mesh: M_ii = h1 h2 h3 / 8 * w_a w_b w_c, doubled per direction on shared faces."""
    p, nc, hi = 3, (2, 3, 2), (1.0, 3.0, 4.0)
    m = orc.Mesh(nc, p, "periodic", (0, 0, 0), hi)
    w = np.array([1 / 6, 5 / 6, 5 / 6, 1 / 6])
    per = [np.tile(np.array([2 * w[0], w[1], w[2]]) * (hi[d] / nc[d]) / 2, nc[d]) for d in range(3)]
    expect = np.einsum("k,j,i->kji", per[2], per[1], per[0]).ravel()
    assert np.allclose(orc.lumped_mass_diagonal(m), expect, rtol=1e-14, atol=0)


# ------------------------------------------------------------------ M^kappa with kappa at the quadrature points
def test_kappa_constant_array_equals_sigma():
    m = _perturbed_mesh(3, "dirichlet")
    a = orc.Operator(m, 2.5)
    b = orc.Operator(m, 0.0, kappa=np.full((12, 64), 2.5))
    X = inputs.multivector(3, m.ndof, 3)
    assert np.array_equal(a.apply(X), b.apply(X))


def test_kappa_moments_closed_form():
    """kappa = 1 + 2x + 3y - z + xy on [0,a]x[0,b]x[0,c], uniform cells: 1^T M^kappa 1 = int kappa and
    x_d^T M^kappa 1 = int kappa x_d (nodal interpolation of x_d is exact; Gauss rule exact).  A kappa array indexed
    with q1 and q3 swapped, or cells in another order, changes the x and z moments."""
    a, b, c = 1.0, 2.0, 1.5
    m = orc.Mesh((3, 2, 2), 2, "natural", (0, 0, 0), (a, b, c))
    xq = orc.quadrature_point_coordinates(m)
    kap = 1 + 2 * xq[..., 0] + 3 * xq[..., 1] - xq[..., 2] + xq[..., 0] * xq[..., 1]
    op = orc.Operator(m, 0.0, ck=0.0, cm=1.0, kappa=kap)
    r = op.apply(np.ones(m.ndof))
    V = a * b * c
    I0 = V * (1 + a + 1.5 * b - 0.5 * c + a * b / 4)
    Ix = V * (a / 2 + 2 * a * a / 3 + 3 * a * b / 4 - a * c / 4 + a * a * b / 6)
    Iy = V * (b / 2 + a * b / 2 + b * b - b * c / 4 + a * b * b / 6)
    Iz = V * (c / 2 + a * c / 2 + 3 * b * c / 4 - c * c / 3 + a * b * c / 8)
    X = m.node_coordinates()
    assert abs(r.sum() - I0) < 1e-13 * I0
    for d, I in enumerate((Ix, Iy, Iz)):
        assert abs(X[:, d] @ r - I) < 1e-13 * I


def test_kappa_operator_is_symmetric_and_matches_dense_element_matrix():
    m = _perturbed_mesh(2, "natural", ncells=(2, 1, 1))
    rng = np.random.default_rng(5)
    kap = rng.uniform(-1, 2, size=(2, 27))
    op = orc.Operator(m, 0.0, ck=0.5, kappa=kap)
    A = op.apply(np.eye(m.ndof))
    assert np.allclose(A, A.T, atol=1e-13)
    # the kappa part alone is N^T diag(kappa det J w) N cell by cell
    Mk = orc.Operator(m, 0.0, ck=0.0, kappa=kap).apply(np.eye(m.ndof))
    K = orc.Operator(m, 0.0, ck=0.5).apply(np.eye(m.ndof))
    assert np.allclose(A, K + Mk, atol=1e-13)
    # independent tables for p = 2: nodes -1, 0, 1, library Gauss points, Lagrange basis written out
    xg, wg = np.polynomial.legendre.leggauss(3)
    N1 = np.stack([xg * (xg - 1) / 2, 1 - xg * xg, xg * (xg + 1) / 2], 1)          # [q][i]
    Nf = np.einsum("ck,bj,ai->cbakji", N1, N1, N1).reshape(27, 27)
    W = np.einsum("c,b,a->cba", wg, wg, wg).ravel()
    ref = np.zeros_like(Mk)
    for e in range(2):
        idx, _ = m.cell_dofs(e, 0, 0)
        v = m.cell_vertices(e, 0, 0)
        det = np.zeros(27)
        for Q in range(27):
            xi = np.array([xg[Q % 3], xg[(Q // 3) % 3], xg[Q // 9]])
            J = np.zeros((3, 3))
            for k in range(8):
                s = np.array([2 * (k & 1) - 1, 2 * ((k >> 1) & 1) - 1, 2 * ((k >> 2) & 1) - 1])
                for d in range(3):
                    g = s[d] / 8.0
                    for o in range(3):
                        if o != d:
                            g *= 1 + s[o] * xi[o]
                    J[:, d] += v[k] * g
            det[Q] = np.linalg.det(J)
        ref[np.ix_(idx, idx)] += Nf.T @ np.diag(kap[e] * det * W) @ Nf
    assert np.allclose(Mk, ref, atol=1e-14)


# ------------------------------------------------------------------ H~ = M^-1/2 (K + M^kappa) M^-1/2
def test_mass_scaled_p1_fourier_modes_closed_form():
    """p = 1, uniform periodic mesh, kappa = 0: K = sum_d K1 x M1 x M1 (trilinear elements), lumped M = h1 h2 h3 I, so
    the Fourier mode exp(i theta.j) is an eigenvector of H~ with eigenvalue
    mu/(h1 h2 h3) sum_d k1(theta_d) prod_{e != d} m1(theta_e),  k1 = (2 - 2 cos theta)/h,  m1 = h (4 + 2 cos theta)/6."""
    nc, hi, mu = (4, 3, 5), (1.0, 1.5, 2.0), 0.5
    m = orc.Mesh(nc, 1, "periodic", (0, 0, 0), hi)
    op = orc.Operator(m, 0.0, ck=mu)
    d = 1.0 / np.sqrt(orc.lumped_mass_diagonal(m))
    h = [hi[k] / nc[k] for k in range(3)]
    jz, jy, jx = np.meshgrid(np.arange(nc[2]), np.arange(nc[1]), np.arange(nc[0]), indexing="ij")
    for kx, ky, kz in [(1, 0, 0), (0, 1, 2), (3, 2, 1), (2, 1, 4)]:
        th = [2 * np.pi * kx / nc[0], 2 * np.pi * ky / nc[1], 2 * np.pi * kz / nc[2]]
        k1 = [(2 - 2 * np.cos(th[k])) / h[k] for k in range(3)]
        m1 = [h[k] * (4 + 2 * np.cos(th[k])) / 6 for k in range(3)]
        lam = mu * (k1[0] * m1[1] * m1[2] + m1[0] * k1[1] * m1[2] + m1[0] * m1[1] * k1[2]) / (h[0] * h[1] * h[2])
        v = np.cos(th[0] * jx + th[1] * jy + th[2] * jz).ravel()
        assert np.allclose(op.apply_mass_scaled(v, d), lam * v, atol=1e-12 * max(lam, 1.0))


def test_mass_scaled_null_vector_and_symmetry():
    """kappa = 0, periodic: H~ M^1/2 1 = 0; H~ is symmetric; multivector form = column by column."""
    m = orc.Mesh((2, 2, 3), 3, "periodic", (0, 0, 0), (1.0, 2.0, 3.0))
    op = orc.Operator(m, 0.0, ck=0.5)
    M = orc.lumped_mass_diagonal(m)
    d = 1.0 / np.sqrt(M)
    assert np.abs(op.apply_mass_scaled(np.sqrt(M), d)).max() < 1e-12
    X = inputs.multivector(11, m.ndof, 4)
    Y = op.apply_mass_scaled(X, d)
    assert np.allclose(Y[:, 2], op.apply_mass_scaled(X[:, 2].copy(), d), rtol=0, atol=1e-12 * np.abs(Y).max())
    assert abs(np.vdot(X[:, 0], Y[:, 1]) - np.vdot(Y[:, 0], X[:, 1])) < 1e-11 * np.abs(Y).max()


def test_mass_scaled_spectrum_converges_to_laplacian():
    """Lowest eigenvalues of H~ (mu = 1/2, kappa = 3 constant through the per-point array) on a periodic cube of side L
    approach mu (2 pi/L)^2 |k|^2 + 3: 0 (x1), 1 (x6), 2 (x12) in units of mu (2 pi/L)^2.  p = 4, 3 cells per direction."""
    L, mu, p, nc = 2.0, 0.5, 4, 3
    m = orc.Mesh((nc,) * 3, p, "periodic", (0, 0, 0), (L,) * 3)
    op = orc.Operator(m, 0.0, ck=mu, kappa=np.full((nc ** 3, (p + 1) ** 3), 3.0))
    d = 1.0 / np.sqrt(orc.lumped_mass_diagonal(m))
    H = op.apply_mass_scaled(np.eye(m.ndof), d)
    ev = np.linalg.eigvalsh((H + H.T) / 2)[:19]
    unit = mu * (2 * np.pi / L) ** 2
    expect = 3.0 + unit * np.array([0] + [1] * 6 + [2] * 12)
    assert np.allclose(ev, expect, rtol=2e-3)
    assert abs(ev[0] - 3.0) < 1e-10
