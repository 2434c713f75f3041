"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times: X is filled on the
device by the seeded generator, the CUDA path runs the whole multivector, and the oracle computes SAMPLED
outputs one by one (rows of Y via the <= 8 cells that touch a node; for the Chebyshev config whole columns,
which are independent).  Bar: |Y_gpu - Y_orc| <= 1e-12 * max|Y_orc| on every sampled entry."""
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
    binding.lib()
    return torch, orc, binding


def sample_nodes(w, count, seed):
    """Seeded sample that always contains corners, an edge, face and wrap/boundary-adjacent nodes."""
    nd = w.nd
    rng = np.random.default_rng(seed)
    pts = [(0, 0, 0), (nd[0] - 1, nd[1] - 1, nd[2] - 1), (w.p, w.p, w.p), (w.p, 1, 2), (nd[0] - 1, 3, w.p),
           (1, 1, 1), (nd[0] - 2, nd[1] - 2, nd[2] - 2), (2 * w.p, nd[1] - 1, 0), (w.p * (w.ncells[0] - 1), 5, 7)]
    pts += [tuple(int(rng.integers(0, nd[d])) for d in range(3)) for _ in range(count - len(pts))]
    return np.array([x + nd[0] * (y + nd[1] * z) for x, y, z in pts], dtype=np.int64)


def oracle_op(orc, w):
    bc = "periodic" if w.bc == inputs.BC_PERIODIC else "dirichlet"
    return orc.Operator(orc.Mesh(w.ncells, w.p, bc, w.box_lo, w.box_hi, vertices=inputs.workload_vertices(w)), w.sigma)


def run_full_apply(env, w, nvec, nsamples=24):
    torch, orc, binding = env
    op = binding.FeMf.from_workload(w)
    X = torch.empty(w.ndof * nvec, dtype=torch.float64, device="cuda")
    Y = torch.full_like(X, float("nan"))
    binding.fill_uniform(X, w.seed)
    op.apply(X, Y, nvec)
    torch.cuda.synchronize()
    Yv = Y.view(w.ndof, nvec)
    scale = float(Yv.abs().max().item())
    assert np.isfinite(scale) and scale > 0
    nodes = sample_nodes(w, nsamples, 17)
    Yo = oracle_op(orc, w).apply_at_nodes(lambda idx: inputs.multivector(w.seed, w.ndof, nvec, rows=idx), nodes)
    Yg = Yv[torch.from_numpy(nodes).cuda()].cpu().numpy()
    err = float(np.abs(Yg - Yo).max() / scale)
    assert err <= TOL, (w.name, nvec, err)
    # property that holds at any size: symmetry u^T (A v) = v^T (A u) with v = a second seeded block
    V = torch.empty_like(X); AV = torch.empty_like(X)
    binding.fill_uniform(V, w.seed + 1000)
    op.apply(V, AV, nvec); torch.cuda.synchronize()
    a = float((X * AV).sum().item()); b = float((V * Y).sum().item())
    assert abs(a - b) <= 1e-10 * max(abs(a), abs(b), 1.0)
    return err


def test_cfg2_full(env):
    w = inputs.configs()[2]
    run_full_apply(env, w, w.nvec)


def test_cfg3_full(env):
    w = inputs.configs()[3]
    run_full_apply(env, w, w.nvec, nsamples=12)


@pytest.mark.parametrize("nvec", [1, 8, 16, 32, 64])
def test_cfg4_full_sweep(env, nvec):
    run_full_apply(env, inputs.configs()[4], nvec, nsamples=12)


def test_cfg5_full_chebyshev(env):
    """All 1024 columns are filtered on the GPU (m = 20); 3 sampled columns are filtered by the oracle on the
    full mesh (columns are independent), with b from the oracle's 10-step Lanczos bound."""
    torch, orc, binding = env
    w = inputs.configs()[5]
    oo = oracle_op(orc, w)
    b = orc.lanczos_upper_bound(oo.apply, inputs.uniform_pm1(inputs.SEED_BASE + 5 + 200, 0, w.ndof), 10)
    assert 2.2 < b < 3.2                                          # DESIGN.md reading 12 (lambda_max ~ 2.16)
    op = binding.FeMf.from_workload(w)
    X = torch.empty(w.ndof * w.nvec, dtype=torch.float64, device="cuda")
    Y = torch.empty_like(X)
    binding.fill_uniform(X, w.seed)
    cols = [0, 517, 1023]
    Xc = X.view(w.ndof, w.nvec)[:, cols].cpu().numpy()
    op.cheb_filter(X, Y, w.nvec, w.cheb_m, w.cheb_a, b, w.cheb_a0)
    torch.cuda.synchronize()
    Yg = Y.view(w.ndof, w.nvec)[:, cols].cpu().numpy()
    Yo = orc.chebyshev_filter(oo.apply, Xc, w.cheb_m, w.cheb_a, b, w.cheb_a0)
    err = float(np.abs(Yg - Yo).max() / np.abs(Yo).max())
    assert err <= TOL, err


# ---------------------------------------------------------------- SURVEY.md 8(f) NEXT-1 at full size
def run_full_eigen_operator(env, w, nvec, nsamples=12):
    """H~ = M^-1/2 (K + M^kappa) M^-1/2 with a seeded kappa per quadrature point, whole multivector on the GPU,
    sampled rows from the oracle: (H~ X)[J] = d_J (H (d.X))[J]."""
    torch, orc, binding = env
    op = binding.FeMf.from_workload(w)
    ncell = w.ncells[0] * w.ncells[1] * w.ncells[2]
    kap = inputs.kappa_points(w.seed + 300, ncell, (w.p + 1) ** 3)
    op.set_kappa(kap)
    op.set_mass_scaling(True)
    X = torch.empty(w.ndof * nvec, dtype=torch.float64, device="cuda")
    Y = torch.full_like(X, float("nan"))
    binding.fill_uniform(X, w.seed)
    op.apply(X, Y, nvec)
    torch.cuda.synchronize()
    Yv = Y.view(w.ndof, nvec)
    scale = float(Yv.abs().max().item())
    assert np.isfinite(scale) and scale > 0
    bc = "periodic" if w.bc == inputs.BC_PERIODIC else "dirichlet"
    mesh = orc.Mesh(w.ncells, w.p, bc, w.box_lo, w.box_hi, vertices=inputs.workload_vertices(w))
    oo = orc.Operator(mesh, 0.0, kappa=kap)
    Mo = orc.lumped_mass_diagonal(mesh)
    # det J comes from differences of vertex coordinates: rounding is amplified by |x| / h (<= cells per direction)
    assert (np.abs(op.mass_diagonal() - Mo) / Mo).max() <= 16 * np.finfo(float).eps * max(w.ncells)
    d = 1.0 / np.sqrt(Mo)
    nodes = sample_nodes(w, nsamples, 23)
    rows = lambda idx: d[idx, None] * inputs.multivector(w.seed, w.ndof, nvec, rows=idx)
    Yo = d[nodes, None] * oo.apply_at_nodes(rows, nodes)
    Yg = Yv[torch.from_numpy(nodes).cuda()].cpu().numpy()
    err = float(np.abs(Yg - Yo).max() / scale)
    assert err <= TOL, (w.name, nvec, op.kernel_name(nvec), err)
    V = torch.empty_like(X); AV = torch.empty_like(X)
    binding.fill_uniform(V, w.seed + 1000)
    op.apply(V, AV, nvec); torch.cuda.synchronize()
    a = float((X * AV).sum().item()); b = float((V * Y).sum().item())
    assert abs(a - b) <= 1e-10 * max(abs(a), abs(b), 1.0)
    return op.kernel_name(nvec)


def test_cfg2_full_eigen_operator(env):
    w = inputs.configs()[2]
    assert run_full_eigen_operator(env, w, w.nvec) == "fe_apply_cart_plane"


def test_cfg4_full_eigen_operator(env):
    w = inputs.configs()[4]
    assert run_full_eigen_operator(env, w, 16) == "fe_apply_cart_line"


def test_cfg3_full_eigen_operator(env):
    w = inputs.configs()[3]
    assert run_full_eigen_operator(env, w, w.nvec, nsamples=10) == "fe_apply_gen_tma"


# ---------------------------------------------------------------- element-by-element at full size
# A persistent kernel with a dynamic work counter can fail LOCALLY (an item skipped or done twice) where a handful of
# sampled nodes will not look: the cases below compare EVERY row of the full-size result.  Two oracles: the cell-matrix
# oracle (fe_oracle.Operator.apply) and, on the uniform Cartesian configs, the exactly integrated Kronecker closed form
# (kron_oracle.kronecker_apply), which shares nothing with the first.
def full_compare(Yg, Yo, what):
    scale = float(np.abs(Yo).max())
    err = float(np.abs(Yg - Yo).max() / scale)
    worst_col = max(float(np.abs(Yg[:, j] - Yo[:, j]).max() / np.abs(Yo[:, j]).max()) for j in range(Yo.shape[1]))
    assert err <= TOL, (what, err, worst_col)
    return err


@pytest.mark.parametrize("nvec", [1, 8])
def test_cfg4_full_every_row_two_oracles(env, nvec):
    """Config 4 (p = 7, 32^3 periodic cells, 11.2 M DoFs) at nvec 1 (cells-as-slots kernel) and 8 (line kernel)."""
    torch, orc, binding = env
    from oracle import kron_oracle as kro
    w = inputs.configs()[4]
    op = binding.FeMf.from_workload(w)
    X = torch.empty(w.ndof * nvec, dtype=torch.float64, device="cuda")
    Y = torch.full_like(X, float("nan"))
    binding.fill_uniform(X, w.seed)
    op.apply(X, Y, nvec); torch.cuda.synchronize()
    Xh = X.cpu().numpy().reshape(w.ndof, nvec)
    Yg = Y.cpu().numpy().reshape(w.ndof, nvec)
    Yk = kro.kronecker_apply(w.ncells, w.p, "periodic", w.box_lo, w.box_hi, w.sigma, Xh)
    full_compare(Yg, Yk, ("cfg4 kron", nvec, op.kernel_name(nvec)))
    Yo = oracle_op(orc, w).apply(Xh)
    full_compare(Yg, Yo, ("cfg4 cell-matrix", nvec, op.kernel_name(nvec)))


def test_cfg3_full_every_row_four_columns(env):
    """Config 3 (p = 8, perturbed mesh, per-q-point metric): the GPU applies all 16 columns, the cell-matrix oracle the
    first, two middle and last column on the full mesh; every row of those columns is compared."""
    torch, orc, binding = env
    w = inputs.configs()[3]
    nvec = w.nvec
    op = binding.FeMf.from_workload(w)
    X = torch.empty(w.ndof * nvec, dtype=torch.float64, device="cuda")
    Y = torch.full_like(X, float("nan"))
    binding.fill_uniform(X, w.seed)
    op.apply(X, Y, nvec); torch.cuda.synchronize()
    cols = [0, 5, 10, 15]
    Xc = np.ascontiguousarray(X.view(w.ndof, nvec)[:, cols].cpu().numpy())
    Yg = Y.view(w.ndof, nvec)[:, cols].cpu().numpy()
    assert np.isfinite(Y.cpu().numpy()).all()
    Yo = oracle_op(orc, w).apply(Xc)
    full_compare(Yg, Yo, ("cfg3", op.kernel_name(nvec)))


def test_cfg5_full_apply_every_row_eight_columns(env):
    """Config 5's mesh and block (p = 6, 16^3 periodic cells on [0,10]^3, 1024 vectors = 64 vector blocks of the plane
    kernel): a single apply of the whole block, 8 columns spread over the vector blocks compared on every row."""
    torch, orc, binding = env
    from oracle import kron_oracle as kro
    w = inputs.configs()[5]
    nvec = w.nvec
    op = binding.FeMf.from_workload(w)
    X = torch.empty(w.ndof * nvec, dtype=torch.float64, device="cuda")
    Y = torch.full_like(X, float("nan"))
    binding.fill_uniform(X, w.seed)
    op.apply(X, Y, nvec); torch.cuda.synchronize()
    assert op.kernel_name(nvec) == "fe_apply_cart_plane"
    cols = [0, 15, 16, 300, 517, 800, 1008, 1023]
    Xc = np.ascontiguousarray(X.view(w.ndof, nvec)[:, cols].cpu().numpy())
    Yg = Y.view(w.ndof, nvec)[:, cols].cpu().numpy()
    Yk = kro.kronecker_apply(w.ncells, w.p, "periodic", w.box_lo, w.box_hi, w.sigma, Xc)
    full_compare(Yg, Yk, "cfg5 kron")
    Yo = oracle_op(orc, w).apply(Xc)
    full_compare(Yg, Yo, "cfg5 cell-matrix")
    # the other 1016 columns: finite, and the column sums of K X vanish on a periodic mesh (K 1 = 0), i.e.
    # 1^T (A X) = sigma 1^T M X = sigma * (cell volume weights) -- checked against the Kronecker row sums
    (Mx, _), (My, _), (Mz, _) = kro.matrices_1d(w.ncells, w.p, "periodic", w.box_lo, w.box_hi)
    wgt = np.einsum("k,j,i->kji", Mz.sum(0), My.sum(0), Mx.sum(0)).reshape(-1)
    lhs = Y.view(w.ndof, nvec).sum(0).cpu().numpy()
    rhs = w.sigma * (torch.from_numpy(wgt).cuda()[:, None] * X.view(w.ndof, nvec)).sum(0).cpu().numpy()
    assert np.isfinite(lhs).all()
    assert np.abs(lhs - rhs).max() <= 1e-9 * max(np.abs(rhs).max(), 1.0)


def test_cfg2_full_every_row_kronecker(env):
    """Config 2 (the bench workload, Dirichlet): all 32 columns, every row, against the Kronecker closed form (the
    cell-matrix oracle is compared on the full block inside bench.py's cpu_baseline leg)."""
    torch, orc, binding = env
    from oracle import kron_oracle as kro
    w = inputs.configs()[2]
    nvec = w.nvec
    op = binding.FeMf.from_workload(w)
    X = torch.empty(w.ndof * nvec, dtype=torch.float64, device="cuda")
    Y = torch.full_like(X, float("nan"))
    binding.fill_uniform(X, w.seed)
    op.apply(X, Y, nvec); torch.cuda.synchronize()
    Xh = X.cpu().numpy().reshape(w.ndof, nvec)
    Yg = Y.cpu().numpy().reshape(w.ndof, nvec)
    Yk = kro.kronecker_apply(w.ncells, w.p, "dirichlet", w.box_lo, w.box_hi, w.sigma, Xh)
    full_compare(Yg, Yk, "cfg2 kron")
