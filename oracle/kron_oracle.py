"""Second CPU oracle for UNIFORM CARTESIAN meshes -- TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as fe_oracle.py:
only tests/, smoke() and bench.py's cpu_baseline legs may import it; it imports nothing from the package).

On a uniform box with constant coefficients the operator of PAPER.md:71-77 (Eq. 3) / PAPER.md:99-106 (Eq. 6) separates
("Affine Cartesian meshes -- closed form"):

    A = Mz (x) My (x) Kx  +  Mz (x) Ky (x) Mx  +  Kz (x) My (x) Mx  +  sigma Mz (x) My (x) Mx

with the ASSEMBLED 1-D mass / stiffness matrices of the degree-p Lagrange basis on the GLL nodes (periodic wrap,
or rows and columns of the two boundary nodes zeroed for homogeneous Dirichlet = C^T A C, reading 7).  Gauss
quadrature with n_q = p + 1 points integrates these degree-2p integrands exactly, so this is the same operator as
the one fe_oracle.Operator assembles from 3-D element matrices -- reached by a route that shares nothing with it:
no 3-D tables, no element matrices, no gather/scatter; its own Lagrange evaluation (product formulas in float64)
and numpy's Gauss-Legendre rule with p + 3 points.  The only thing taken from fe_oracle is the GLL node positions
(themselves pinned against the roots of P'_p).

Cheap enough to run at BASELINE.json's full sizes (7 mode products of nd^4 nvec flops each), where it serves as an
element-by-element check of the CUDA path beside fe_oracle.Operator.apply.

Pins (tests/test_oracle_kron.py, -m "not gpu"): textbook 1-D matrices for p = 1, 2; row sums
(K 1 = 0, 1^T M 1 = length); agreement with fe_oracle.Operator.apply on anisotropic periodic / Dirichlet meshes for
p up to 8; exact energies of separable polynomials.
"""
from __future__ import annotations

import numpy as np

from . import fe_oracle as _fe


def lagrange_1d(nodes: np.ndarray, x: np.ndarray):
    """L[q, i] = l_i(x_q) and dL[q, i] = l_i'(x_q) by the product / sum-of-products formulas."""
    n = len(nodes)
    L = np.ones((len(x), n))
    dL = np.zeros((len(x), n))
    for i in range(n):
        for j in range(n):
            if j != i:
                L[:, i] *= (x - nodes[j]) / (nodes[i] - nodes[j])
        for k in range(n):
            if k == i:
                continue
            term = np.full(len(x), 1.0 / (nodes[i] - nodes[k]))
            for j in range(n):
                if j != i and j != k:
                    term *= (x - nodes[j]) / (nodes[i] - nodes[j])
            dL[:, i] += term
    return L, dL


def element_matrices_1d(p: int, h: float):
    """(M_e, K_e) of one cell of length h: M_e[i,j] = int l_i l_j dx, K_e[i,j] = int l_i' l_j' dx, by numpy's
    Gauss-Legendre rule with p + 3 points (exact up to degree 2p + 5 >= 2p)."""
    xi = np.asarray(_fe.gll_nodes(p), dtype=np.float64)
    xg, wg = np.polynomial.legendre.leggauss(p + 3)
    L, dL = lagrange_1d(xi, xg)
    M = (L * wg[:, None]).T @ L * (h / 2.0)
    K = (dL * wg[:, None]).T @ dL * (2.0 / h)
    return 0.5 * (M + M.T), 0.5 * (K + K.T)


def assemble_1d(Ae: np.ndarray, ncell: int, p: int, bc: str) -> np.ndarray:
    """Global 1-D matrix: cells overlap in one node; periodic wraps, dirichlet zeroes the boundary rows / columns."""
    nd = ncell * p + (0 if bc == "periodic" else 1)
    A = np.zeros((nd, nd))
    for e in range(ncell):
        idx = (e * p + np.arange(p + 1)) % nd
        A[np.ix_(idx, idx)] += Ae
    if bc == "dirichlet":
        A[0, :] = A[-1, :] = 0.0
        A[:, 0] = A[:, -1] = 0.0
    return A


def matrices_1d(ncells, p: int, bc: str, box_lo, box_hi):
    out = []
    for d in range(3):
        Me, Ke = element_matrices_1d(p, (box_hi[d] - box_lo[d]) / ncells[d])
        out.append((assemble_1d(Me, ncells[d], p, bc), assemble_1d(Ke, ncells[d], p, bc)))
    return out


def kronecker_apply(ncells, p: int, bc: str, box_lo, box_hi, sigma: float, X: np.ndarray) -> np.ndarray:
    """Y = A X for X of shape (ndof, nvec), node index x fastest (the layout of every multivector in this repo)."""
    (Mx, Kx), (My, Ky), (Mz, Kz) = matrices_1d(ncells, p, bc, box_lo, box_hi)
    ndx, ndy, ndz = Mx.shape[0], My.shape[0], Mz.shape[0]
    nvec = X.shape[1]
    assert X.shape[0] == ndx * ndy * ndz
    X4 = np.ascontiguousarray(X, dtype=np.float64).reshape(ndz, ndy, ndx, nvec)

    def mode_x(A, T):   # (A T)[z, y, :, v]
        return np.matmul(A, T.reshape(ndz * ndy, ndx, nvec)).reshape(ndz, ndy, ndx, nvec)

    def mode_y(A, T):
        return np.matmul(A, T.reshape(ndz, ndy, ndx * nvec)).reshape(ndz, ndy, ndx, nvec)

    def mode_z(A, T):
        return (A @ T.reshape(ndz, ndy * ndx * nvec)).reshape(ndz, ndy, ndx, nvec)

    mx = mode_x(Mx, X4)
    kx = mode_x(Kx, X4)
    t3 = mode_y(My, mx)                               # My Mx X
    t12 = mode_y(My, kx) + mode_y(Ky, mx) + sigma * t3
    Y = mode_z(Mz, t12) + mode_z(Kz, t3)
    return Y.reshape(ndx * ndy * ndz, nvec)
