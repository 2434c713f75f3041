"""CPU oracle for the hot path of arXiv 2208.07129 -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference`
legs may import this file.  It shares no code with the CUDA path (`paper_2208_07129_b200/csrc`)
and imports nothing from the package.

What it computes (the plain definition, Eq. 3, Eq. 6,
PAPER.md:108-128 Eq. 7-9): Y = A X with A = K + sigma*M assembled from DENSE element matrices
obtained by full tensor Gauss quadrature -- the paper's "cell-matrix" method in its most
literal form.  No sum factorisation, no D = D~N factorisation, no sqrt(w)
rescaling, no even-odd decomposition.  numpy float64 throughout; the 1D nodes,
weights and Lagrange tables are computed in x87 long double and rounded once.  `A @ U`
(a library matmul) is used as one step, as the cell-matrix method prescribes.

Readings of silent / garbled passages are those of SURVEY.md §8(c) (listed in DESIGN.md §3).

Pins (tests/test_oracle_pins.py, `-m "not gpu"`): 1D-table identities, textbook p=1/p=2
element matrices, exactly integrated Kronecker closed form on Cartesian meshes, symmetry,
K*1 = 0, 1^T M 1 = |Omega|, exact polynomial energies, patch test on the perturbed mesh,
long-double brute force on a single cell, Chebyshev closed form T_m, Lanczos bound >= lambda_max,
the paper's printed DoF counts.  Nothing here is "parity unpinned".

SURVEY.md §8(f) NEXT-1 pieces (pins in tests/test_oracle_mass_scaled.py): kappa given at the quadrature points
(`Operator(kappa=...)`), the GLL-lumped mass diagonal (`lumped_mass_diagonal`) and
H~ = M^-1/2 (K + M^kappa) M^-1/2 (`Operator.apply_mass_scaled`, Eq. B.1).  Pinned by
printed Lobatto weights, the rule's exactness, sum M_ii = |Omega|, lumped = row sums of the consistent mass,
closed-form moments of a bilinear kappa, the p = 1 Fourier closed form and the Laplacian spectrum on a periodic cube.
"""
from __future__ import annotations

import numpy as np

LD = np.longdouble

# --------------------------------------------------------------------------------------
# 1D data  (PAPER.md:54, 158 GLL nodes; PAPER.md:117 quadrature)
# --------------------------------------------------------------------------------------


def _legendre(n: int, x):
    """P_n(x) and P_{n-1}(x) by the three-term recurrence, long double."""
    x = np.asarray(x, dtype=LD)
    p0 = np.ones_like(x)
    if n == 0:
        return p0, np.zeros_like(x)
    p1 = x.copy()
    for k in range(2, n + 1):
        p0, p1 = p1, ((2 * k - 1) * x * p1 - (k - 1) * p0) / LD(k)
    return p1, p0


def _legendre_d1_d2(n: int, x):
    """P_n, P_n', P_n'' at interior points |x| < 1 (Legendre ODE for the second derivative)."""
    pn, pnm1 = _legendre(n, x)
    d1 = LD(n) * (x * pn - pnm1) / (x * x - LD(1))
    d2 = (LD(2) * x * d1 - LD(n) * LD(n + 1) * pn) / (LD(1) - x * x)
    return pn, d1, d2


def gll_nodes(p: int) -> np.ndarray:
    """p+1 Gauss-Legendre-Lobatto nodes on [-1,1]: +-1 and the roots of P'_p (long double)."""
    if p < 1:
        raise ValueError("p >= 1")
    x = -np.cos(np.pi * np.arange(p + 1, dtype=LD) / LD(p))
    xi = x[1:-1].copy()
    for _ in range(100):
        _, d1, d2 = _legendre_d1_d2(p, xi)
        dx = d1 / d2
        xi = xi - dx
        if np.max(np.abs(dx), initial=LD(0)) < LD(1e-19):
            break
    x[1:-1] = xi
    x[0], x[-1] = LD(-1), LD(1)
    # enforce exact anti-symmetry of the node set
    x = (x - x[::-1]) / LD(2)
    return x


def gll_weights(p: int) -> np.ndarray:
    """Weights of the (p+1)-point Gauss-Lobatto-Legendre rule: w_i = 2 / (p (p+1) P_p(xi_i)^2) (long double)."""
    x = gll_nodes(p)
    pn, _ = _legendre(p, x)
    w = LD(2) / (LD(p) * LD(p + 1) * pn * pn)
    return (w + w[::-1]) / LD(2)


def gauss_legendre(n: int):
    """n-point Gauss-Legendre points and weights on [-1,1] (long double)."""
    k = np.arange(n, dtype=LD)
    x = -np.cos(LD(np.pi) * (k + LD(0.75)) / (LD(n) + LD(0.5)))
    for _ in range(100):
        pn, pnm1 = _legendre(n, x)
        d1 = LD(n) * (x * pn - pnm1) / (x * x - LD(1))
        dx = pn / d1
        x = x - dx
        if np.max(np.abs(dx)) < LD(1e-19):
            break
    x = (x - x[::-1]) / LD(2)
    pn, pnm1 = _legendre(n, x)
    d1 = LD(n) * (x * pn - pnm1) / (x * x - LD(1))
    w = LD(2) / ((LD(1) - x * x) * d1 * d1)
    w = (w + w[::-1]) / LD(2)
    return x, w


def lagrange_values(nodes, x):
    """L[q][i] = l_i(x_q) for the Lagrange basis on `nodes` (long double, product formula)."""
    nodes = np.asarray(nodes, dtype=LD)
    x = np.asarray(x, dtype=LD)
    n = len(nodes)
    L = np.ones((len(x), n), dtype=LD)
    for i in range(n):
        for j in range(n):
            if j != i:
                L[:, i] *= (x - nodes[j]) / (nodes[i] - nodes[j])
    return L


def lagrange_derivatives(nodes, x):
    """D[q][i] = l_i'(x_q): sum over k != i of 1/(x_i-x_k) * prod_{j != i,k} (x-x_j)/(x_i-x_j)."""
    nodes = np.asarray(nodes, dtype=LD)
    x = np.asarray(x, dtype=LD)
    n = len(nodes)
    D = np.zeros((len(x), n), dtype=LD)
    for i in range(n):
        for k in range(n):
            if k == i:
                continue
            term = np.full(len(x), LD(1) / (nodes[i] - nodes[k]), dtype=LD)
            for j in range(n):
                if j != i and j != k:
                    term *= (x - nodes[j]) / (nodes[i] - nodes[j])
            D[:, i] += term
    return D


def tables_1d(p: int, nq: int | None = None):
    """(xi, xq, w, N1, D1) as float64: N1[q][i] = l_i(xq_q), D1[q][i] = l_i'(xq_q) on GLL nodes xi,
    Gauss-Legendre points xq / weights w, n_q = p+1 by default (SURVEY.md §8(c) readings 1-2)."""
    nq = p + 1 if nq is None else nq
    xi = gll_nodes(p)
    xq, w = gauss_legendre(nq)
    N1 = lagrange_values(xi, xq)
    D1 = lagrange_derivatives(xi, xq)
    f = lambda a: np.asarray(a, dtype=np.float64)
    return f(xi), f(xq), f(w), f(N1), f(D1)


def collocation_derivative_1d(p: int, nq: int | None = None) -> np.ndarray:
    """D~[q][r] = l~_r'(xq_q), Lagrange basis on the QUADRATURE points.
    Not used by the oracle's apply; exists for the pin D1 = D~ N1."""
    nq = p + 1 if nq is None else nq
    xq, _ = gauss_legendre(nq)
    return np.asarray(lagrange_derivatives(xq, xq), dtype=np.float64)


# --------------------------------------------------------------------------------------
# 3D reference tables (Eq. 10, Eq. 11)
# --------------------------------------------------------------------------------------


def tables_3d(p: int, nq: int | None = None):
    """Dense Nf[Q][I], Df[s][Q][I] (s = 0,1,2) and W[Q] with I = i1 + n i2 + n^2 i3 (Eq. 18 order,
    PAPER.md:308) and Q = q1 + n q2 + n^2 q3."""
    _, _, w, N1, D1 = tables_1d(p, nq)
    # np.kron(A, B)[a*nb + b', ...]: the LEFT factor carries the slowest index.
    Nf = np.kron(N1, np.kron(N1, N1))
    Df = np.stack([
        np.kron(N1, np.kron(N1, D1)),   # d/dxi_1 (fastest index)
        np.kron(N1, np.kron(D1, N1)),   # d/dxi_2
        np.kron(D1, np.kron(N1, N1)),   # d/dxi_3 (slowest index)
    ])
    W = np.kron(w, np.kron(w, w))
    return Nf, Df, W


def reference_points_3d(p: int, nq: int | None = None):
    """(n^3, 3) quadrature points in Q order and (n^3, 3) GLL nodes in I order."""
    xi, xq, _, _, _ = tables_1d(p, nq)
    n = p + 1
    nq = n if nq is None else nq
    q = np.arange(nq ** 3)
    q1, q2, q3 = q % nq, (q // nq) % nq, q // (nq * nq)
    i = np.arange(n ** 3)
    i1, i2, i3 = i % n, (i // n) % n, i // (n * n)
    return np.stack([xq[q1], xq[q2], xq[q3]], 1), np.stack([xi[i1], xi[i2], xi[i3]], 1)


# --------------------------------------------------------------------------------------
# Geometry (PAPER.md:92 reference cell [-1,1]^3; Eq. 7b-c)
# --------------------------------------------------------------------------------------

_CORNER_SIGNS = np.array([[2 * (v & 1) - 1, 2 * ((v >> 1) & 1) - 1, 2 * ((v >> 2) & 1) - 1] for v in range(8)],
                         dtype=np.float64)


def trilinear_map(verts8: np.ndarray, pts: np.ndarray):
    """x(xi) (npts,3) and J[a][c] = dx_a/dxi_c (npts,3,3) of the trilinear map whose vertex
    v = v1 + 2 v2 + 4 v3 sits at reference corner (2v1-1, 2v2-1, 2v3-1)."""
    s = _CORNER_SIGNS
    f = 0.5 * (1.0 + s[None, :, :] * pts[:, None, :])          # (npts, 8, 3) factors (1 + s xi)/2
    phi = f[:, :, 0] * f[:, :, 1] * f[:, :, 2]
    x = phi @ verts8
    J = np.zeros((pts.shape[0], 3, 3))
    for c in range(3):
        o = [d for d in range(3) if d != c]
        dphi = 0.5 * s[None, :, c] * f[:, :, o[0]] * f[:, :, o[1]]   # d phi_v / d xi_c
        J[:, :, c] = dphi @ verts8
    return x, J


def geometric_factors(verts8: np.ndarray, qpts: np.ndarray, W: np.ndarray, sigma):
    """G[s][d][Q] = (J^-1 J^-T)_sd det J w_Q (mu = 1) and g[Q] = kappa_Q det J w_Q (Eq. 22
    PAPER.md:336-341): sigma is the constant kappa of the Helmholtz operator or an array kappa_Q of n_q^3 values."""
    _, J = trilinear_map(verts8, qpts)
    det = np.linalg.det(J)
    if np.any(det <= 0.0):
        raise ValueError("non-positive det J")
    Jinv = np.linalg.inv(J)
    Ginv = np.einsum("qsa,qda->qsd", Jinv, Jinv)                   # J^-1 J^-T
    G = np.transpose(Ginv * (det * W)[:, None, None], (1, 2, 0))     # (3,3,nq3)
    g = sigma * det * W
    return G, g


def element_matrix(Nf, Df, G, g) -> np.ndarray:
    """A_e = sum_{s,d} Df[s]^T diag(G[s][d]) Df[d] + Nf^T diag(g) Nf  (Eq. 8, 9)."""
    A = Nf.T @ (g[:, None] * Nf)
    for s in range(3):
        for d in range(3):
            A += Df[s].T @ (G[s][d][:, None] * Df[d])
    return A


def element_apply_dense(Nf, Df, G, g, U) -> np.ndarray:
    """The same expression applied right-to-left to U (n^3 x nvec) with the DENSE 3D tables
    (full quadrature, no sum factorisation) -- used when every cell has its own geometry."""
    T = Nf @ U
    Td = [Df[d] @ U for d in range(3)]
    V = Nf.T @ (g[:, None] * T)
    for s in range(3):
        S = G[s][0][:, None] * Td[0] + G[s][1][:, None] * Td[1] + G[s][2][:, None] * Td[2]
        V += Df[s].T @ S
    return V


# --------------------------------------------------------------------------------------
# Mesh and index maps (readings 7 and 9; Eq. 18)
# --------------------------------------------------------------------------------------


class Mesh:
    """Structured hexahedral mesh of ncells = (ncx, ncy, ncz) cells, degree p.

    bc: "periodic" (nd = N p, indices wrap), "dirichlet" (nd = N p + 1, boundary nodes read as 0
    and written as 0: C^T A C literally, reading 7) or "natural" (nd = N p + 1,
    no constraint; only used by the pins).  vertices: None for the uniform Cartesian mesh of
    [box_lo, box_hi], else an array [(ncz+1)][(ncy+1)][(ncx+1)][3]."""

    def __init__(self, ncells, p, bc, box_lo=(0.0, 0.0, 0.0), box_hi=(1.0, 1.0, 1.0), vertices=None):
        if bc not in ("periodic", "dirichlet", "natural"):
            raise ValueError(bc)
        self.ncells = tuple(int(c) for c in ncells)
        self.p = int(p)
        self.n = self.p + 1
        self.bc = bc
        self.box_lo = tuple(float(v) for v in box_lo)
        self.box_hi = tuple(float(v) for v in box_hi)
        self.vertices = None if vertices is None else np.asarray(vertices, dtype=np.float64)
        add = 0 if bc == "periodic" else 1
        self.nd = tuple(c * self.p + add for c in self.ncells)
        self.ndof = self.nd[0] * self.nd[1] * self.nd[2]
        if bc == "periodic" and min(self.ncells) < 2:
            raise ValueError("periodic needs >= 2 cells per direction")
        n = self.n
        I = np.arange(n ** 3)
        self._i = (I % n, (I // n) % n, I // (n * n))

    def cell_vertices(self, ex, ey, ez) -> np.ndarray:
        """(8,3) vertices of cell (ex,ey,ez), vertex v = v1 + 2 v2 + 4 v3."""
        if self.vertices is not None:
            return np.array([self.vertices[ez + ((v >> 2) & 1), ey + ((v >> 1) & 1), ex + (v & 1)] for v in range(8)])
        h = [(self.box_hi[d] - self.box_lo[d]) / self.ncells[d] for d in range(3)]
        e = (ex, ey, ez)
        return np.array([[self.box_lo[d] + h[d] * (e[d] + ((v >> d) & 1)) for d in range(3)] for v in range(8)])

    def cell_dofs(self, ex, ey, ez):
        """Global indices g(e, I) (n^3,) and a mask of Dirichlet-boundary nodes."""
        p, nd = self.p, self.nd
        ix, iy, iz = ex * p + self._i[0], ey * p + self._i[1], ez * p + self._i[2]
        if self.bc == "periodic":
            ix, iy, iz = ix % nd[0], iy % nd[1], iz % nd[2]
            mask = None
        elif self.bc == "dirichlet":
            mask = ((ix == 0) | (ix == nd[0] - 1) | (iy == 0) | (iy == nd[1] - 1) | (iz == 0) | (iz == nd[2] - 1))
        else:
            mask = None
        return ix + nd[0] * (iy + nd[1] * iz), mask

    def node_coordinates(self) -> np.ndarray:
        """(ndof, 3) physical coordinates of the global nodes (isoparametric image of the GLL nodes)."""
        _, gl = reference_points_3d(self.p)
        out = np.zeros((self.ndof, 3))
        for ez in range(self.ncells[2]):
            for ey in range(self.ncells[1]):
                for ex in range(self.ncells[0]):
                    idx, _ = self.cell_dofs(ex, ey, ez)
                    x, _ = trilinear_map(self.cell_vertices(ex, ey, ez), gl)
                    out[idx] = x
        return out


def quadrature_point_coordinates(mesh: Mesh, nq: int | None = None) -> np.ndarray:
    """(ncells, n_q^3, 3) physical coordinates x_Q^(e) of the quadrature points, cells in
    lexicographic order (x fastest), Q = q1 + n q2 + n^2 q3."""
    qp, _ = reference_points_3d(mesh.p, nq)
    ncx, ncy, ncz = mesh.ncells
    out = np.zeros((ncx * ncy * ncz, qp.shape[0], 3))
    for ez in range(ncz):
        for ey in range(ncy):
            for ex in range(ncx):
                out[ex + ncx * (ey + ncy * ez)], _ = trilinear_map(mesh.cell_vertices(ex, ey, ez), qp)
    return out


def lumped_mass_diagonal(mesh: Mesh) -> np.ndarray:
    """diag(M) with the overlap integrals evaluated by the GLL rule on the nodes themselves:
    M_ii = sum over the cells that contain node i of det J(xi_i) w_i1 w_i2 w_i3.  Dirichlet boundary nodes keep
    their entry (they are masked by the operator anyway)."""
    w1 = gll_weights(mesh.p).astype(np.float64)
    n = mesh.n
    I = np.arange(n ** 3)
    w3 = w1[I % n] * w1[(I // n) % n] * w1[I // (n * n)]
    _, gl = reference_points_3d(mesh.p)
    M = np.zeros(mesh.ndof)
    for ez in range(mesh.ncells[2]):
        for ey in range(mesh.ncells[1]):
            for ex in range(mesh.ncells[0]):
                idx, _ = mesh.cell_dofs(ex, ey, ez)
                _, J = trilinear_map(mesh.cell_vertices(ex, ey, ez), gl)
                np.add.at(M, idx, np.linalg.det(J) * w3)
    return M


class Operator:
    """A = K + sigma*M on a Mesh by the cell-matrix method (PAPER.md:134-143 steps 1-4).

    split=(ck, cm) scales the stiffness and mass parts (pins use (1,0) and (0,1)); the default is
    K + sigma M."""

    def __init__(self, mesh: Mesh, sigma: float, ck: float = 1.0, cm: float = 1.0, form_matrices: bool = False,
                 kappa=None, nq: int | None = None):
        """kappa: None (constant sigma) or an array [ncells][n_q^3] of values at the quadrature points of every cell
        (cells in lexicographic order, x fastest; Eq. 22, the "precomputed potential" of
        PAPER.md:796), which then replaces sigma.  nq: Gauss points per direction, n_p = p + 1 by default; the paper
        also benchmarks n_q = n_p + 2."""
        self.mesh, self.sigma, self.ck, self.cm = mesh, float(sigma), float(ck), float(cm)
        self.nq = mesh.p + 1 if nq is None else int(nq)      # points per direction; n_p + 2 = over-integration (NEXT-2)
        self.kappa = None if kappa is None else np.asarray(kappa, dtype=np.float64).reshape(
            mesh.ncells[0] * mesh.ncells[1] * mesh.ncells[2], self.nq ** 3)
        self.Nf, self.Df, self.W = tables_3d(mesh.p, self.nq)
        self.qpts, _ = reference_points_3d(mesh.p, self.nq)
        self.form_matrices = form_matrices
        self._Ae_uniform = None
        if mesh.vertices is None and self.kappa is None:
            # every cell of a uniform Cartesian mesh has the same A_e: a property of the input
            self._Ae_uniform = self.cell_matrix(0, 0, 0)

    def _factors(self, ex, ey, ez):
        kap = self.sigma
        if self.kappa is not None:
            kap = self.kappa[ex + self.mesh.ncells[0] * (ey + self.mesh.ncells[1] * ez)]
        G, g = geometric_factors(self.mesh.cell_vertices(ex, ey, ez), self.qpts, self.W, kap)
        return self.ck * G, self.cm * g

    def cell_matrix(self, ex, ey, ez) -> np.ndarray:
        if self._Ae_uniform is not None:
            return self._Ae_uniform
        G, g = self._factors(ex, ey, ez)
        return element_matrix(self.Nf, self.Df, G, g)

    def cell_apply(self, ex, ey, ez, U) -> np.ndarray:
        if self._Ae_uniform is not None:
            return self._Ae_uniform @ U
        G, g = self._factors(ex, ey, ez)
        if self.form_matrices:
            return element_matrix(self.Nf, self.Df, G, g) @ U
        return element_apply_dense(self.Nf, self.Df, G, g, U)

    def apply(self, X: np.ndarray) -> np.ndarray:
        """Y = A X, X of shape (ndof, nvec) (vector index innermost).  Fixed cell order (z, y, x)."""
        m = self.mesh
        X = np.asarray(X, dtype=np.float64)
        if X.ndim == 1:
            return self.apply(X[:, None])[:, 0]
        if X.shape[0] != m.ndof:
            raise ValueError("X has %d rows, mesh has %d dofs" % (X.shape[0], m.ndof))
        Y = np.zeros_like(X)
        for ez in range(m.ncells[2]):
            for ey in range(m.ncells[1]):
                for ex in range(m.ncells[0]):
                    idx, mask = m.cell_dofs(ex, ey, ez)
                    U = X[idx]                                   # Q^(e): extraction
                    if mask is not None:
                        U[mask] = 0.0                            # C: boundary nodes read as 0
                    V = self.cell_apply(ex, ey, ez, U)           # A^(e) U^(e)
                    if mask is not None:
                        V[mask] = 0.0                            # C^T: boundary rows dropped
                    Y[idx] += V                                  # Q^(e)T: assembly (idx unique per cell)
        return Y

    def apply_mass_scaled(self, X: np.ndarray, d: np.ndarray) -> np.ndarray:
        """H~ X = M^-1/2 (K + M^kappa) M^-1/2 X with d = diag(M)^-1/2 of the GLL-lumped mass matrix
        (Eq. 26; Eq. B.1 PAPER.md:1171 with a = 1, b = c = 0)."""
        X = np.asarray(X, dtype=np.float64)
        if X.ndim == 1:
            return d * self.apply(d * X)
        return d[:, None] * self.apply(d[:, None] * X)

    def apply_at_nodes(self, x_rows, nodes) -> np.ndarray:
        """Rows `nodes` of Y = A X without forming X: x_rows(idx) must return X[idx] (len(idx), nvec).
        Visits only the (<= 8) cells that contain each node.  Used for sampled full-size parity."""
        m = self.mesh
        p, nd, nc = m.p, m.nd, m.ncells
        out = []
        for J in np.asarray(nodes, dtype=np.int64):
            jx, jy, jz = int(J % nd[0]), int((J // nd[0]) % nd[1]), int(J // (nd[0] * nd[1]))
            cells = [[], [], []]
            for d, j in enumerate((jx, jy, jz)):
                for e in range(nc[d]):
                    for i in range(p + 1):
                        gi = e * p + i
                        if m.bc == "periodic":
                            gi %= nd[d]
                        if gi == j:
                            cells[d].append(e)
                cells[d] = sorted(set(cells[d]))
            acc = None
            for ez in cells[2]:
                for ey in cells[1]:
                    for ex in cells[0]:
                        idx, mask = m.cell_dofs(ex, ey, ez)
                        U = np.array(x_rows(idx), dtype=np.float64)
                        if mask is not None:
                            U[mask] = 0.0
                        V = self.cell_apply(ex, ey, ez, U)
                        if mask is not None:
                            V[mask] = 0.0
                        rows = np.nonzero(idx == J)[0]
                        contrib = V[rows].sum(axis=0)
                        acc = contrib if acc is None else acc + contrib
            out.append(acc)
        return np.array(out)


# --------------------------------------------------------------------------------------
# Chebyshev filter (Alg. 6 lines 2-17, reading 10)
# --------------------------------------------------------------------------------------


def to_bcv(X: np.ndarray, b: int) -> np.ndarray:
    """Batched Contiguous Vector layout (section 3.2.1, Fig. 1): "stores the nodal values of a batch of b
    vectors contiguously for all nodes in n_b = ceil(n_v / b) contiguous batches".  X [ndof][nvec] -> flat array, batch
    after batch, each batch [ndof][b_i] with the vector index innermost (the last batch holds the remaining vectors)."""
    X = np.asarray(X, dtype=np.float64)
    return np.concatenate([np.ascontiguousarray(X[:, v0:v0 + b]).reshape(-1) for v0 in range(0, X.shape[1], b)])


def from_bcv(flat: np.ndarray, ndof: int, nvec: int, b: int) -> np.ndarray:
    """Inverse of to_bcv."""
    flat = np.asarray(flat, dtype=np.float64).reshape(-1)
    X = np.empty((ndof, nvec))
    for v0 in range(0, nvec, b):
        bi = min(b, nvec - v0)
        X[:, v0:v0 + bi] = flat[ndof * v0:ndof * (v0 + bi)].reshape(ndof, bi)
    return X


def chebyshev_filter(apply, X: np.ndarray, m: int, a: float, b: float, a0: float) -> np.ndarray:
    """Scaled Chebyshev filter of degree m damping [a, b], a0 = lower spectral bound.
    Temporaries named as in the paper: e, c, sigma, sigma1, gamma, alpha1, alpha2."""
    if m < 1 or not (b > a) or not (a0 < a):
        raise ValueError("need m >= 1, b > a, a0 < a")
    e = (b - a) / 2.0
    c = (b + a) / 2.0
    sigma = e / (a0 - c)
    sigma1 = sigma
    gamma = 2.0 / sigma1
    alpha1 = sigma1 / e
    alpha2 = -c
    X = np.array(X, dtype=np.float64)
    Y = alpha1 * apply(X) + (alpha1 * alpha2) * X            # Y <- a1 H X + a1 a2 X
    for _ in range(2, m + 1):
        sigma2 = 1.0 / (gamma - sigma)
        alpha1 = 2.0 * sigma2 / e
        alpha2 = -sigma * sigma2
        Xn = alpha1 * apply(Y) + alpha2 * X - (c * alpha1) * Y
        X, Y = Y, Xn                                          # swap(X, Y)
        sigma = sigma2
    return Y


def lanczos_upper_bound(apply, v0: np.ndarray, k: int = 10) -> float:
    """k-step plain Lanczos bound lambda_max(T_k) + beta_k (Zhou-Saad [37])."""
    v = np.asarray(v0, dtype=np.float64)
    v = v / np.linalg.norm(v)
    v_prev = np.zeros_like(v)
    beta = 0.0
    alphas, betas = [], []
    for _ in range(k):
        w = apply(v) - beta * v_prev
        alpha = float(v @ w)
        w = w - alpha * v
        beta = float(np.linalg.norm(w))
        alphas.append(alpha)
        betas.append(beta)
        if beta == 0.0:
            break
        v_prev, v = v, w / beta
    T = np.diag(alphas) + np.diag(betas[:-1], 1) + np.diag(betas[:-1], -1)
    return float(np.linalg.eigvalsh(T)[-1] + betas[-1])


# --------------------------------------------------------------------------------------
# Chebyshev filtered subspace iteration (Alg. 6)
# --------------------------------------------------------------------------------------

def chfsi_iterate(apply, U: np.ndarray, m: int, lam_max: float, lam_u: float, lam_min: float, free=None):
    """One pass of Alg. 6 lines 2-20: filter U with degree m damping [lam_u, lam_max] (lines 2-17), orthogonalise the
    filtered block (line 18; any orthonormal basis of its span: Householder QR here), solve the projected problem
    Xo^T H Xo Q = Q Lambda (line 19) and rotate U = Xo Q (line 20).  Returns (U, Lambda ascending, residual norms
    ||H u_j - lambda_j u_j||_2 of line 1).

    free: boolean mask of the unconstrained rows (None: all).  With C^T A C (reading 7) every constrained DoF is a
    null vector of H~, i.e. an eigenvalue 0 inside the wanted interval; the eigenproblem is posed on the unconstrained
    DoFs, so the subspace must keep exact zeros in the constrained rows.  The filter and the rotation do; a Householder
    QR of the whole block would not (it mixes rows at rounding level, which later passes amplify), hence the
    orthogonalisation acts on the free rows."""
    Y = chebyshev_filter(apply, U, m, lam_u, lam_max, lam_min)
    if free is None:
        Xo, _ = np.linalg.qr(Y)
    else:
        Xo = np.zeros_like(Y)
        Xo[free], _ = np.linalg.qr(Y[free])
    HX = apply(Xo)
    T = Xo.T @ HX
    lam, Q = np.linalg.eigh((T + T.T) / 2.0)
    Un = Xo @ Q
    R = apply(Un) - Un * lam[None, :]
    return Un, lam, np.linalg.norm(R, axis=0)


def chfsi_solve(apply, U0: np.ndarray, n_wanted: int, m: int, lam_max: float, lam_u: float, lam_min: float,
                tau: float, max_iter: int = 50, free=None):
    """Alg. 6 line 1 loop: repeat chfsi_iterate until the n_wanted lowest pairs have residual <= tau.  The paper takes
    the bounds as data and is silent on how they follow the iteration; reading (Zhou-Saad [37]): after
    each pass lam_min <- lowest Ritz value, lam_u <- highest Ritz value of the subspace (the vectors beyond n_wanted
    are the buffer).  Returns (U, Lambda, residuals, passes)."""
    U = np.array(U0, dtype=np.float64)
    if free is not None:
        U[~free] = 0.0
    lam = res = None
    for it in range(1, max_iter + 1):
        U, lam, res = chfsi_iterate(apply, U, m, lam_max, lam_u, lam_min, free)
        if res[:n_wanted].max() <= tau:
            return U, lam, res, it
        lam_min, lam_u = float(lam[0]), float(lam[-1])
    return U, lam, res, max_iter
