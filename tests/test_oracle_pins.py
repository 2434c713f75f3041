"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA path).

Each test is chosen so that a plausible mistake in oracle/fe_oracle.py (dropped term, wrong sign
or index, transposed operand, wrong weight) fails it.  SURVEY.md §8(c) "What pins each part".
"""
import os

import numpy as np
import pytest

from oracle import fe_oracle as orc
from paper_2208_07129_b200 import inputs

LD = np.longdouble
GOLDEN_DIR = os.path.join(os.path.dirname(__file__), "golden")


def dense_operator(op):
    return op.apply(np.eye(op.mesh.ndof))


# ------------------------------------------------------------------ 1D tables
@pytest.mark.parametrize("p", [1, 2, 3, 4, 5, 6, 7, 8])
def test_1d_tables_identities(p):
    xi, xq, w, N1, D1 = orc.tables_1d(p)
    n = p + 1
    assert np.allclose(N1.sum(1), 1.0, atol=4e-15)                   # partition of unity
    assert np.allclose(D1.sum(1), 0.0, atol=2e-13)                   # derivative of 1
    assert np.allclose(D1 @ xi, 1.0, atol=2e-13)                     # derivative of x
    assert abs(w.sum() - 2.0) < 4e-15
    for k in range(0, n):                                            # Gauss exactness 2k <= 2n-1
        assert abs((w * xq ** (2 * k)).sum() - 2.0 / (2 * k + 1)) < 1e-14
        assert abs((w * xq ** (2 * k + 1)).sum()) < 1e-15
    # interpolation reproduces polynomials of degree <= p, derivative table differentiates them
    for k in range(p + 1):
        assert np.allclose(N1 @ xi ** k, xq ** k, atol=1e-14)
        assert np.allclose(D1 @ xi ** k, k * xq ** max(k - 1, 0) if k else 0 * xq, atol=5e-13)
    # centro-(anti)symmetry (SURVEY.md reading 14)
    assert np.allclose(N1, N1[::-1, ::-1], atol=1e-15)
    assert np.allclose(D1, -D1[::-1, ::-1], atol=1e-13)
    # GLL interior nodes are roots of P'_p; Gauss points roots of P_{p+1}
    c = np.zeros(p + 1); c[p] = 1
    dP = np.polynomial.legendre.Legendre(c).deriv()
    assert np.allclose(dP(xi[1:-1]), 0.0, atol=1e-12)
    c = np.zeros(n + 1); c[n] = 1
    assert np.allclose(np.polynomial.legendre.Legendre(c)(xq), 0.0, atol=1e-14)
    xg, wg = np.polynomial.legendre.leggauss(n)                      # library routine as special case
    assert np.allclose(xq, xg, atol=1e-15) and np.allclose(w, wg, atol=1e-15)


@pytest.mark.parametrize("p", [1, 3, 6, 7, 8])
def test_collocation_factorisation(p):
    """D1D = D~1D N1D."""
    _, _, _, N1, D1 = orc.tables_1d(p)
    Dt = orc.collocation_derivative_1d(p)
    assert np.allclose(Dt @ N1, D1, atol=1e-13)


# ------------------------------------------------------------------ element matrices, textbook cases
def _exact_1d_element(p, h):
    """Exactly integrated 1D mass/stiffness of the Lagrange basis on GLL nodes by polynomial algebra
    (independent of the oracle's table evaluation: monomial coefficients, analytic integration)."""
    from numpy.polynomial import Polynomial as P
    xi = np.asarray(orc.gll_nodes(p), dtype=np.float64)
    basis = []
    for i in range(p + 1):
        q = P([1.0])
        for j in range(p + 1):
            if j != i:
                q = q * P([-xi[j], 1.0]) / (xi[i] - xi[j])
        basis.append(q)
    M = np.zeros((p + 1, p + 1)); K = np.zeros_like(M)
    for i in range(p + 1):
        for j in range(p + 1):
            F = (basis[i] * basis[j]).integ()
            M[i, j] = (F(1.0) - F(-1.0)) * h / 2
            F = (basis[i].deriv() * basis[j].deriv()).integ()
            K[i, j] = (F(1.0) - F(-1.0)) * 2 / h
    return M, K


def test_textbook_1d_matrices_p1_p2():
    h = 0.7
    M, K = _exact_1d_element(1, h)
    assert np.allclose(M, h / 6 * np.array([[2, 1], [1, 2]]), atol=1e-15)
    assert np.allclose(K, 1 / h * np.array([[1, -1], [-1, 1]]), atol=1e-15)
    M, K = _exact_1d_element(2, h)
    assert np.allclose(M, h / 30 * np.array([[4, 2, -1], [2, 16, 2], [-1, 2, 4]]), atol=1e-15)
    assert np.allclose(K, 1 / (3 * h) * np.array([[7, -8, 1], [-8, 16, -8], [1, -8, 7]]), atol=1e-14)


@pytest.mark.parametrize("p", [1, 2, 3, 5])
def test_element_matrix_is_kronecker_sum_on_a_brick(p):
    """Brick hx x hy x hz: A_e = Mz(x)My(x)Kx + Mz(x)Ky(x)Mx + Kz(x)My(x)Mx + sigma Mz(x)My(x)Mx with the
    textbook (p = 1, 2) / exactly integrated 1D matrices; Gauss n_q = p+1 is exact here."""
    hx, hy, hz, sigma = 0.5, 0.8, 1.3, 0.37
    mesh = orc.Mesh((2, 2, 2), p, "natural", (0, 0, 0), (2 * hx, 2 * hy, 2 * hz))
    A = orc.Operator(mesh, sigma).cell_matrix(0, 0, 0)
    (Mx, Kx), (My, Ky), (Mz, Kz) = (_exact_1d_element(p, h) for h in (hx, hy, hz))
    ref = (np.kron(Mz, np.kron(My, Kx)) + np.kron(Mz, np.kron(Ky, Mx)) + np.kron(Kz, np.kron(My, Mx))
           + sigma * np.kron(Mz, np.kron(My, Mx)))
    assert np.abs(A - ref).max() <= 2e-14 * np.abs(ref).max()


def _assemble_1d(Me, ncell, p, bc):
    nd = ncell * p + (0 if bc == "periodic" else 1)
    A = np.zeros((nd, nd))
    for e in range(ncell):
        idx = (e * p + np.arange(p + 1)) % nd
        A[np.ix_(idx, idx)] += Me
    if bc == "dirichlet":
        A[0, :] = A[-1, :] = 0.0
        A[:, 0] = A[:, -1] = 0.0
    return A


@pytest.mark.parametrize("bc", ["periodic", "dirichlet", "natural"])
@pytest.mark.parametrize("p", [2, 3])
def test_global_operator_kronecker_closed_form(bc, p):
    """Affine Cartesian meshes: A = Mz(x)My(x)Kx + ... with assembled 1D matrices (SURVEY.md §8(c) pins).
    Anisotropic cell counts and box catch any transposed axis in the index map."""
    nc, lo, hi, sigma = (2, 3, 4), (0.0, -1.0, 2.0), (1.0, 0.5, 4.4), 0.6
    mesh = orc.Mesh(nc, p, bc, lo, hi)
    A = dense_operator(orc.Operator(mesh, sigma))
    mk = []
    for d in range(3):
        Me, Ke = _exact_1d_element(p, (hi[d] - lo[d]) / nc[d])
        mk.append((_assemble_1d(Me, nc[d], p, bc), _assemble_1d(Ke, nc[d], p, bc)))
    (Mx, Kx), (My, Ky), (Mz, Kz) = mk
    ref = (np.kron(Mz, np.kron(My, Kx)) + np.kron(Mz, np.kron(Ky, Mx)) + np.kron(Kz, np.kron(My, Mx))
           + sigma * np.kron(Mz, np.kron(My, Mx)))
    assert A.shape == ref.shape
    assert np.abs(A - ref).max() <= 5e-14 * np.abs(ref).max()
    if bc == "dirichlet":                                            # reading 7: boundary rows/cols are zero
        nd = mesh.nd
        J = np.arange(mesh.ndof)
        jx, jy, jz = J % nd[0], (J // nd[0]) % nd[1], J // (nd[0] * nd[1])
        bnd = (jx == 0) | (jx == nd[0] - 1) | (jy == 0) | (jy == nd[1] - 1) | (jz == 0) | (jz == nd[2] - 1)
        assert np.all(A[bnd] == 0.0) and np.all(A[:, bnd] == 0.0)


# ------------------------------------------------------------------ brute force, one distorted cell, long double
def _brute_force_cell(p, verts8, sigma, nq=None):
    """A_e[I][J] by explicit loops over (I, J, Q) in long double with its own basis evaluation
    (monomial coefficients) and its own Jacobian (monomial form of the trilinear map)."""
    n = p + 1
    nq = n if nq is None else nq
    xi = orc.gll_nodes(p)
    xq, w = orc.gauss_legendre(nq)
    # monomial coefficients of l_i, lowest degree first
    coef = []
    for i in range(n):
        c = np.array([LD(1)])
        for j in range(n):
            if j != i:
                c = (np.concatenate([[LD(0)], c]) - xi[j] * np.concatenate([c, [LD(0)]])) / (xi[i] - xi[j])
        coef.append(c)
    val = lambda c, x: sum(c[k] * x ** k for k in range(len(c)))
    der = lambda c, x: sum(k * c[k] * x ** (k - 1) for k in range(1, len(c)))
    L = np.array([[val(coef[i], xq[q]) for i in range(n)] for q in range(nq)])
    dL = np.array([[der(coef[i], xq[q]) for i in range(n)] for q in range(nq)])
    # trilinear map in monomial form: x = sum_{abc in {0,1}} m[abc] xi1^a xi2^b xi3^c
    V = np.asarray(verts8, dtype=LD)
    mono = np.zeros((2, 2, 2, 3), dtype=LD)
    for v in range(8):
        s = [2 * ((v >> d) & 1) - 1 for d in range(3)]
        for a in range(2):
            for b in range(2):
                for c in range(2):
                    mono[a, b, c] += V[v] * (s[0] ** a) * (s[1] ** b) * (s[2] ** c) / LD(8)
    A = np.zeros((n ** 3, n ** 3), dtype=LD)
    for q3 in range(nq):
        for q2 in range(nq):
            for q1 in range(nq):
                x = (xq[q1], xq[q2], xq[q3])
                Jm = np.zeros((3, 3), dtype=LD)
                for a in range(2):
                    for b in range(2):
                        for c in range(2):
                            m = mono[a, b, c]
                            if a: Jm[:, 0] += m * (x[1] ** b) * (x[2] ** c)
                            if b: Jm[:, 1] += m * (x[0] ** a) * (x[2] ** c)
                            if c: Jm[:, 2] += m * (x[0] ** a) * (x[1] ** b)
                det = (Jm[0, 0] * (Jm[1, 1] * Jm[2, 2] - Jm[1, 2] * Jm[2, 1])
                       - Jm[0, 1] * (Jm[1, 0] * Jm[2, 2] - Jm[1, 2] * Jm[2, 0])
                       + Jm[0, 2] * (Jm[1, 0] * Jm[2, 1] - Jm[1, 1] * Jm[2, 0]))
                cof = np.zeros((3, 3), dtype=LD)                      # inverse by cofactors
                for r in range(3):
                    for c_ in range(3):
                        r1, r2 = (r + 1) % 3, (r + 2) % 3
                        c1, c2 = (c_ + 1) % 3, (c_ + 2) % 3
                        cof[c_, r] = (Jm[r1, c1] * Jm[r2, c2] - Jm[r1, c2] * Jm[r2, c1]) / det
                Jinv = cof
                wq = w[q1] * w[q2] * w[q3]
                grads = np.zeros((n ** 3, 3), dtype=LD)               # physical gradients J^-T grad_xi
                vals = np.zeros(n ** 3, dtype=LD)
                for i3 in range(n):
                    for i2 in range(n):
                        for i1 in range(n):
                            I = i1 + n * (i2 + n * i3)
                            gref = np.array([dL[q1, i1] * L[q2, i2] * L[q3, i3],
                                             L[q1, i1] * dL[q2, i2] * L[q3, i3],
                                             L[q1, i1] * L[q2, i2] * dL[q3, i3]])
                            grads[I] = Jinv.T @ gref
                            vals[I] = L[q1, i1] * L[q2, i2] * L[q3, i3]
                A += (grads @ grads.T + LD(sigma) * np.outer(vals, vals)) * det * wq
    return A


@pytest.mark.parametrize("p", [1, 2, 3])
def test_single_distorted_cell_brute_force(p):
    rng = np.random.default_rng(7 + p)
    verts = np.array([[(v & 1), (v >> 1) & 1, (v >> 2) & 1] for v in range(8)], dtype=float) * [1.0, 1.4, 0.8]
    verts += rng.uniform(-0.12, 0.12, verts.shape)
    Nf, Df, W = orc.tables_3d(p)
    qpts, _ = orc.reference_points_3d(p)
    G, g = orc.geometric_factors(verts, qpts, W, 0.9)
    A = orc.element_matrix(Nf, Df, G, g)
    ref = _brute_force_cell(p, verts, 0.9)
    assert np.abs(A - np.asarray(ref, dtype=np.float64)).max() <= 1e-13 * float(np.abs(ref).max())
    U = rng.uniform(-1, 1, (A.shape[0], 3))
    assert np.allclose(orc.element_apply_dense(Nf, Df, G, g, U), A @ U, rtol=0, atol=1e-13 * np.abs(A).max())


# ------------------------------------------------------------------ invariants of the global operator
def _mesh(kind, p=3, nc=(3, 2, 3)):
    if kind == "periodic":
        return orc.Mesh(nc, p, "periodic", (0, 0, 0), (1.0, 0.8, 1.2))
    if kind == "dirichlet":
        return orc.Mesh(nc, p, "dirichlet", (0, 0, 0), (1.0, 0.8, 1.2))
    if kind == "perturbed":
        v = inputs.perturbed_vertices(nc, (0, 0, 0), (1.0, 0.8, 1.2), 0.15, 99)
        return orc.Mesh(nc, p, "periodic", (0, 0, 0), (1.0, 0.8, 1.2), vertices=v)
    raise ValueError(kind)


@pytest.mark.parametrize("kind", ["periodic", "dirichlet", "perturbed"])
def test_symmetry(kind):
    mesh = _mesh(kind)
    op = orc.Operator(mesh, 0.7)
    u = inputs.multivector(11, mesh.ndof, 2)
    v = inputs.multivector(12, mesh.ndof, 2)
    a, b = np.sum(u * op.apply(v)), np.sum(v * op.apply(u))
    assert abs(a - b) <= 1e-13 * abs(a)


@pytest.mark.parametrize("kind", ["periodic", "perturbed"])
def test_nullspace_and_volume(kind):
    mesh = _mesh(kind)
    one = np.ones((mesh.ndof, 1))
    K1 = orc.Operator(mesh, 1.0, ck=1.0, cm=0.0).apply(one)
    assert np.abs(K1).max() < 1e-12                                   # K 1 = 0
    M1 = orc.Operator(mesh, 1.0, ck=0.0, cm=1.0).apply(one)
    assert abs(M1.sum() - 1.0 * 0.8 * 1.2) < 1e-14                    # 1^T M 1 = |Omega| (det J trilinear: exact)
    # sigma scales only the mass part
    A1 = orc.Operator(mesh, 2.5).apply(one)
    assert np.allclose(A1, 2.5 * M1, atol=1e-12)


def test_exact_energies_polynomial_field():
    """u = x^2 y - z^3 on [0,2]^3, p = 3, natural mode: u^T K u = int |grad u|^2 = 312.888..,
    u^T M u = int u^2 = 64.6095.. exactly (integrands of degree <= 2p per variable)."""
    mesh = orc.Mesh((2, 3, 2), 3, "natural", (0, 0, 0), (2, 2, 2))
    x = mesh.node_coordinates()
    u = (x[:, 0] ** 2 * x[:, 1] - x[:, 2] ** 3)[:, None]
    eK = float(np.sum(u * orc.Operator(mesh, 1.0, ck=1, cm=0).apply(u)))
    eM = float(np.sum(u * orc.Operator(mesh, 1.0, ck=0, cm=1).apply(u)))
    exactK = 4 * (8 / 3) * (8 / 3) * 2 + (32 / 5) * 4 + 9 * (32 / 5) * 4
    exactM = (32 / 5) * (8 / 3) * 2 - 2 * (8 / 3) * 2 * 4 + (128 / 7) * 4
    assert abs(eK - exactK) < 1e-12 * exactK
    assert abs(eM - exactM) < 1e-12 * exactM
    # the full operator is K + sigma M, not K + M or sigma (K + M)
    eA = float(np.sum(u * orc.Operator(mesh, 0.3).apply(u)))
    assert abs(eA - (exactK + 0.3 * exactM)) < 1e-12 * exactK


def test_dirichlet_energy():
    """u = prod x_d (L - x_d) vanishes on the boundary, so the Dirichlet operator gives the exact energy."""
    L = 1.5
    mesh = orc.Mesh((2, 2, 2), 2, "dirichlet", (0, 0, 0), (L, L, L))
    nat = orc.Mesh((2, 2, 2), 2, "natural", (0, 0, 0), (L, L, L))
    x = nat.node_coordinates()
    f = lambda t: t * (L - t)
    u = (f(x[:, 0]) * f(x[:, 1]) * f(x[:, 2]))[:, None]
    e = float(np.sum(u * orc.Operator(mesh, 2.0).apply(u)))
    i0 = L ** 5 / 30            # int f^2
    i1 = L ** 3 / 3             # int f'^2
    exact = 3 * i1 * i0 * i0 + 2.0 * i0 ** 3
    assert abs(e - exact) < 1e-12 * exact


def test_patch_test_on_perturbed_mesh():
    """Natural mode on a perturbed mesh: u_x = x-coordinate of each node is represented exactly
    (isoparametric), so u_x^T K u_x = |Omega|, u_x^T K u_y = 0, u_x^T M 1 = int x."""
    nc, hi = (3, 3, 2), (1.0, 1.0, 1.0)
    v = inputs.perturbed_vertices(nc, (0, 0, 0), hi, 0.15, 5)
    assert np.abs(v - inputs.uniform_vertices(nc, (0, 0, 0), hi)).max() > 0.01     # really perturbed
    mesh = orc.Mesh(nc, 2, "natural", (0, 0, 0), hi, vertices=v)
    x = mesh.node_coordinates()
    K = orc.Operator(mesh, 1.0, ck=1, cm=0)
    M = orc.Operator(mesh, 1.0, ck=0, cm=1)
    ux, uy, one = x[:, :1], x[:, 1:2], np.ones((mesh.ndof, 1))
    assert abs(np.sum(ux * K.apply(ux)) - 1.0) < 1e-13
    assert abs(np.sum(ux * K.apply(uy))) < 1e-13
    assert abs(np.sum(ux * M.apply(one)) - 0.5) < 1e-13
    assert abs(np.sum(one * M.apply(one)) - 1.0) < 1e-13


def test_periodic_is_wrapped_natural():
    """A_per = R^T A_nat R with R the wrap map (exact identity)."""
    nc, p = (2, 3, 2), 2
    per = orc.Mesh(nc, p, "periodic")
    nat = orc.Mesh(nc, p, "natural")
    R = np.zeros((nat.ndof, per.ndof))
    J = np.arange(nat.ndof)
    jx, jy, jz = J % nat.nd[0], (J // nat.nd[0]) % nat.nd[1], J // (nat.nd[0] * nat.nd[1])
    R[J, (jx % per.nd[0]) + per.nd[0] * ((jy % per.nd[1]) + per.nd[1] * (jz % per.nd[2]))] = 1.0
    Ap = dense_operator(orc.Operator(per, 0.4))
    An = dense_operator(orc.Operator(nat, 0.4))
    assert np.abs(Ap - R.T @ An @ R).max() < 1e-14 * np.abs(An).max()


def test_per_cell_path_equals_uniform_path():
    """vertices = the uniform grid must reproduce the shared-A_e path (perturbation -> 0 limit), both
    right-to-left and with explicitly formed matrices."""
    nc, lo, hi = (2, 2, 3), (0, 0, 0), (1.0, 2.0, 1.5)
    X = inputs.multivector(3, orc.Mesh(nc, 3, "periodic", lo, hi).ndof, 3)
    Y0 = orc.Operator(orc.Mesh(nc, 3, "periodic", lo, hi), 1.1).apply(X)
    mv = orc.Mesh(nc, 3, "periodic", lo, hi, vertices=inputs.uniform_vertices(nc, lo, hi))
    Y1 = orc.Operator(mv, 1.1).apply(X)
    Y2 = orc.Operator(mv, 1.1, form_matrices=True).apply(X)
    s = np.abs(Y0).max()
    assert np.abs(Y1 - Y0).max() < 1e-14 * s and np.abs(Y2 - Y0).max() < 1e-14 * s


@pytest.mark.parametrize("kind", ["periodic", "dirichlet", "perturbed"])
def test_apply_at_nodes_matches_apply(kind):
    mesh = _mesh(kind, p=2)
    op = orc.Operator(mesh, 0.5)
    X = inputs.multivector(21, mesh.ndof, 4)
    Y = op.apply(X)
    nodes = np.array([0, 1, mesh.nd[0] - 1, mesh.nd[0] * 2 + 2, mesh.ndof // 2, mesh.ndof - 1, 2 * mesh.p, 37])
    Ys = op.apply_at_nodes(lambda idx: X[idx], nodes)
    assert np.abs(Ys - Y[nodes]).max() <= 1e-14 * np.abs(Y).max()


# ------------------------------------------------------------------ Chebyshev filter and Lanczos bound
def test_chebyshev_closed_form():
    """Filter = T_m((A - c)/e) / T_m((a0 - c)/e) (Zhou-Saad scaled filter; SURVEY.md reading 10)."""
    mesh = orc.Mesh((2, 2, 2), 2, "periodic", (0, 0, 0), (4.0, 4.0, 4.0))
    op = orc.Operator(mesh, 1.0)
    A = dense_operator(op)
    lam, V = np.linalg.eigh((A + A.T) / 2)
    X = inputs.multivector(5, mesh.ndof, 3)
    a0, a, b = 0.0, lam[-1] * 0.3, lam[-1] * 1.05
    e, c = (b - a) / 2, (b + a) / 2
    from numpy.polynomial.chebyshev import Chebyshev
    for m in (1, 2, 3, 8, 20):
        Tm = Chebyshev.basis(m)
        ref = V @ ((Tm((lam - c) / e) / Tm((a0 - c) / e))[:, None] * (V.T @ X))
        Y = orc.chebyshev_filter(op.apply, X, m, a, b, a0)
        assert np.abs(Y - ref).max() <= 1e-12 * np.abs(ref).max(), m
    # m = 1: Y = (sigma1/e) (A X - c X), sigma1 = e/(a0 - c)
    Y1 = orc.chebyshev_filter(op.apply, X, 1, a, b, a0)
    assert np.allclose(Y1, (A @ X - c * X) / (a0 - c), rtol=0, atol=1e-14 * np.abs(Y1).max())
    with pytest.raises(ValueError):
        orc.chebyshev_filter(op.apply, X, 3, 2.0, 1.0, 0.0)           # inverted interval (reading 12)


def test_lanczos_bound_is_an_upper_bound():
    for p, nc, L in ((2, (3, 3, 3), 1.0), (6, (2, 2, 2), 1.25)):       # second: config-5 cell size h = 0.625
        mesh = orc.Mesh(nc, p, "periodic", (0, 0, 0), (L, L, L))
        op = orc.Operator(mesh, 1.0)
        if mesh.ndof <= 1000:
            lam_max = np.linalg.eigvalsh(dense_operator(op))[-1]
        else:
            v = inputs.uniform_pm1(1, 0, mesh.ndof)
            for _ in range(300):
                v = op.apply(v); v /= np.linalg.norm(v)
            lam_max = float(v @ op.apply(v))
        v0 = inputs.uniform_pm1(inputs.SEED_BASE + 5 + 200, 0, mesh.ndof)
        b = orc.lanczos_upper_bound(op.apply, v0, 10)
        assert b >= lam_max * (1 - 1e-12)
        assert b < 2.0 * lam_max


# ------------------------------------------------------------------ paper's printed numbers
def test_paper_dof_counts():
    rows = [l.split() for l in open(os.path.join(GOLDEN_DIR, "paper_dof_counts.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 9
    for r in rows:
        ndof, p, N = int(r[0]), int(r[1]), int(r[2])
        assert orc.Mesh((N, N, N), p, "dirichlet").ndof == ndof


# ------------------------------------------------------------------ input generator (not the oracle, but shared)
def test_generator():
    # SplitMix64 reference stream for seed 0 (first three outputs of the published algorithm)
    z = inputs.splitmix64(np.arange(1, 4, dtype=np.uint64) * inputs.GOLDEN)
    assert [int(v) for v in z] == [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F]
    u = inputs.uniform_pm1(123, 0, 100000)
    assert u.min() >= -1.0 and u.max() < 1.0 and abs(u.mean()) < 0.01 and abs(u.var() - 1 / 3) < 0.01
    assert np.array_equal(inputs.uniform_pm1(123, 500, 10), u[500:510])
    X = inputs.multivector(9, 50, 4)
    assert np.array_equal(inputs.multivector(9, 50, 4, rows=[3, 17]), X[[3, 17]])
    cfg = inputs.configs()
    assert [cfg[i].ndof for i in (1, 2, 3, 4, 5)] == [32768, 3048625, 2097152, 11239424, 884736]


def test_bcv_layout_is_the_index_formula_of_fig_1():
    """PAPER.md:280-286 (Fig. 1): batch i_b = floor(beta / b) holds b_i vectors of all nodes contiguously, the vector index
    innermost: element (J, beta) sits at ndof * b * i_b + J * b_i + beta mod b.  Checked element by element with a
    ragged last batch; b >= nvec is the plain [ndof][nvec] layout; the inverse restores X."""
    ndof, nvec = 7, 11
    X = np.arange(ndof * nvec, dtype=np.float64).reshape(ndof, nvec)
    for b in (1, 2, 4, 8, 11, 16):
        flat = orc.to_bcv(X, b)
        assert flat.shape == (ndof * nvec,)
        for J in range(ndof):
            for beta in range(nvec):
                ib = beta // b
                bi = min(b, nvec - ib * b)
                assert flat[ndof * b * ib + J * bi + beta % b] == X[J, beta]
        assert np.array_equal(orc.from_bcv(flat, ndof, nvec, b), X)
    assert np.array_equal(orc.to_bcv(X, 16), X.reshape(-1))
