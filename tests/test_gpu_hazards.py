"""Regression tests of product hazards found in review (round-1 VERDICT "weak" 8-10): each walks the call
order that used to corrupt memory or results and compares with the CPU oracle."""
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


def bc_name(bc):
    return "periodic" if bc == inputs.BC_PERIODIC else "dirichlet"


def oracle_mesh(orc, w):
    return orc.Mesh(w.ncells, w.p, bc_name(w.bc), w.box_lo, w.box_hi, vertices=inputs.workload_vertices(w))


def relerr(a, b):
    return float(np.abs(a - b).max() / np.abs(b).max())


@pytest.mark.parametrize("p,geom,nvec", [(6, inputs.GEOM_AFFINE, 64), (8, inputs.GEOM_QPOINT, 18), (7, inputs.GEOM_AFFINE, 50)])
def test_apply_host_many_chunks_stress(env, p, geom, nvec):
    """fe_mf_apply_host alternates its column chunks between two internal streams; each stream must own its work
    counter (a counter reset of chunk k+1 under the running persistent kernel of chunk k made items run twice).
    Tiny meshes make the H2D copy as short as the kernel; many repetitions; nvec = 18 gives a 2-column tail chunk."""
    torch, orc, binding = env
    w = inputs.Workload(f"host_stress_p{p}", p, (3, 3, 2), inputs.BC_PERIODIC, geom, 0.9, (0.0, 0.0, 0.0), (1.5, 1.5, 1.0),
                        nvec, 7100 + p, perturb=0.12 if geom == inputs.GEOM_QPOINT else 0.0)
    X = inputs.multivector(w.seed, w.ndof, nvec)
    Yo = orc.Operator(oracle_mesh(orc, w), w.sigma).apply(X)
    op = binding.FeMf.from_workload(w)
    Xh = torch.from_numpy(X).contiguous().pin_memory()
    Yh = torch.empty_like(Xh).pin_memory()
    worst = 0.0
    for rep in range(200):
        Yh.fill_(float("nan"))
        op.apply_host(Xh, Yh, nvec)
        worst = max(worst, relerr(Yh.numpy(), Yo))
    assert worst <= TOL, worst


def test_apply_host_with_caller_work_in_flight(env):
    """The caller's stream keeps launching applies on the context while apply_host runs on the internal streams."""
    torch, orc, binding = env
    w = inputs.Workload("host_inflight", 6, (3, 3, 3), inputs.BC_DIRICHLET, inputs.GEOM_AFFINE, 0.5, (0, 0, 0), (1, 1, 1), 32, 7200)
    X = inputs.multivector(w.seed, w.ndof, w.nvec)
    Yo = orc.Operator(oracle_mesh(orc, w), w.sigma).apply(X)
    op = binding.FeMf.from_workload(w)
    Xd = torch.from_numpy(X).cuda(); Yd = torch.empty_like(Xd)
    Xh = torch.from_numpy(X).contiguous().pin_memory(); Yh = torch.empty_like(Xh).pin_memory()
    for rep in range(50):
        for _ in range(4):
            op.apply(Xd, Yd, w.nvec)
        op.apply_host(Xh, Yh, w.nvec)
        torch.cuda.synchronize()
        assert relerr(Yh.numpy(), Yo) <= TOL
        assert relerr(Yd.cpu().numpy(), Yo) <= TOL


@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_DIRICHLET])
def test_set_kappa_none_after_set_quadrature_keeps_tables(env, bc):
    """Uniform box: set_quadrature(p+3) -> set_kappa(k) -> set_kappa(None) used to free the over-integration tables
    (a pasted line of fe_mf_destroy) and leave them dangling.  Every step is checked against the oracle."""
    torch, orc, binding = env
    p = 4
    w = inputs.Workload("oi_kappa_none", p, (3, 2, 2), bc, inputs.GEOM_AFFINE, 0.7, (0, 0, 0), (1.5, 1.0, 1.0), 8, 7300)
    mesh = oracle_mesh(orc, w)
    X = inputs.multivector(w.seed, w.ndof, w.nvec)
    nq = p + 3
    ncell = 3 * 2 * 2
    kap = inputs.kappa_points(w.seed + 1, ncell, nq ** 3, 0.2, 2.0)
    op = binding.FeMf.from_workload(w)
    Xd = torch.from_numpy(X).cuda(); Yd = torch.empty_like(Xd)

    def check(op_o):
        Yd.fill_(float("nan"))
        op.apply(Xd, Yd, w.nvec); torch.cuda.synchronize()
        assert relerr(Yd.cpu().numpy(), op_o.apply(X)) <= TOL

    op.set_quadrature(nq)
    check(orc.Operator(mesh, w.sigma, nq=nq))
    op.set_kappa(kap)
    check(orc.Operator(mesh, 0.0, kappa=kap, nq=nq))
    op.set_kappa(None)
    check(orc.Operator(mesh, w.sigma, nq=nq))          # used to read freed tables
    op.set_kappa(kap)                                  # a new allocation could land on the freed addresses
    op.set_kappa(None)
    check(orc.Operator(mesh, w.sigma, nq=nq))
    op.set_quadrature(p + 1)                           # used to free the tables a second time
    check(orc.Operator(mesh, w.sigma))
    op.destroy()


def test_kappa_is_dropped_when_the_rule_changes_qpoint_context(env):
    """FE_GEOM_QPOINT context: set_kappa(k) on the default rule writes k det J into the stored factors;
    set_quadrature(p+3) and back to p+1 must leave the constant sigma, not the old kappa (fe_mf.h: 'a kappa array set
    before ... is dropped')."""
    torch, orc, binding = env
    p = 3
    w = inputs.Workload("kappa_roundtrip", p, (2, 3, 2), inputs.BC_PERIODIC, inputs.GEOM_QPOINT, 0.8, (0, 0, 0), (1.0, 1.5, 1.0),
                        6, 7400, perturb=0.1)
    mesh = oracle_mesh(orc, w)
    X = inputs.multivector(w.seed, w.ndof, w.nvec)
    kap = inputs.kappa_points(w.seed + 1, 12, (p + 1) ** 3, 0.2, 2.0)
    op = binding.FeMf.from_workload(w)
    Xd = torch.from_numpy(X).cuda(); Yd = torch.empty_like(Xd)

    def check(op_o):
        Yd.fill_(float("nan"))
        op.apply(Xd, Yd, w.nvec); torch.cuda.synchronize()
        assert relerr(Yd.cpu().numpy(), op_o.apply(X)) <= TOL

    op.set_kappa(kap)
    check(orc.Operator(mesh, 0.0, kappa=kap))
    op.set_quadrature(p + 3)
    check(orc.Operator(mesh, w.sigma, nq=p + 3))
    op.set_quadrature(p + 1)
    check(orc.Operator(mesh, w.sigma))                 # used to apply the old kappa again


@pytest.mark.parametrize("p,geom", [(6, inputs.GEOM_AFFINE), (4, inputs.GEOM_QPOINT), (7, inputs.GEOM_AFFINE)])
def test_pointers_aligned_to_8_bytes_only(env, p, geom):
    """Views offset by one double (8-byte aligned only): Eq. B.1 with beta != 0 and the Chebyshev filter's fallback path
    used to run the 128-bit streaming kernels on them (sticky 'misaligned address' fault)."""
    torch, orc, binding = env
    w = inputs.Workload(f"unaligned_p{p}", p, (2, 2, 3), inputs.BC_PERIODIC, geom, 0.9, (0, 0, 0), (1.0, 1.0, 1.5), 6, 7500 + p,
                        perturb=0.1 if geom == inputs.GEOM_QPOINT else 0.0)
    op_o = orc.Operator(oracle_mesh(orc, w), w.sigma)
    X = inputs.multivector(w.seed, w.ndof, w.nvec)
    Z0 = inputs.multivector(w.seed + 1, w.ndof, w.nvec)
    op = binding.FeMf.from_workload(w)
    n = w.ndof * w.nvec
    bufx = torch.zeros(n + 1, dtype=torch.float64, device="cuda")
    bufz = torch.zeros(n + 1, dtype=torch.float64, device="cuda")
    Xd, Zd = bufx[1:], bufz[1:]
    assert Xd.data_ptr() % 16 == 8 and Zd.data_ptr() % 16 == 8
    Xd.copy_(torch.from_numpy(X).reshape(-1)); Zd.copy_(torch.from_numpy(Z0).reshape(-1))
    op.apply_axpby(0.3, Xd, 0.5, -0.25, Zd, w.nvec); torch.cuda.synchronize()
    Yo = op_o.apply(X)
    assert relerr(Zd.cpu().numpy().reshape(w.ndof, w.nvec), 0.5 * Z0 - 0.25 * X + 0.3 * Yo) <= TOL
    m, a, b, a0 = 5, 1.5, 60.0, -0.2
    Fo = orc.chebyshev_filter(op_o.apply, X, m, a, b, a0)
    Xd.copy_(torch.from_numpy(X).reshape(-1))
    op.cheb_filter(Xd, Zd, w.nvec, m, a, b, a0); torch.cuda.synchronize()
    assert relerr(Zd.cpu().numpy().reshape(w.ndof, w.nvec), Fo) <= TOL


@pytest.mark.parametrize("a,b,a0,m", [(2.0, 2.1, 0.0, 200), (2.0, 2.2, -5.0, 120)])
def test_chebyshev_narrow_interval_does_not_underflow(env, a, b, a0, m):
    """The one-launch-per-step form of the recurrence carries scale factors s_k ~ |sigma sigma_2|^(k/2); with a narrow
    damping interval far from a0 they underflow (0/0 -> NaN in X and Y).  The library must detect this on the host and
    take the unscaled recurrence, whose values stay finite."""
    torch, orc, binding = env
    w = inputs.Workload("cheb_underflow", 4, (2, 2, 2), inputs.BC_PERIODIC, inputs.GEOM_AFFINE, 1.0, (0, 0, 0), (10, 10, 10), 4, 7600)
    op_o = orc.Operator(oracle_mesh(orc, w), w.sigma)
    X = inputs.multivector(w.seed, w.ndof, w.nvec)
    Fo = orc.chebyshev_filter(op_o.apply, X, m, a, b, a0)
    assert np.isfinite(Fo).all()
    op = binding.FeMf.from_workload(w)
    Xd = torch.from_numpy(X).cuda(); Fd = torch.full_like(Xd, float("nan"))
    op.cheb_filter(Xd, Fd, w.nvec, m, a, b, a0); torch.cuda.synchronize()
    F = Fd.cpu().numpy()
    assert np.isfinite(F).all()
    assert np.isfinite(Xd.cpu().numpy()).all()
    assert relerr(F, Fo) <= TOL


@pytest.mark.parametrize("p,bc,geom,nc,nvec", [
    (6, inputs.BC_DIRICHLET, inputs.GEOM_AFFINE, (3, 2, 7), 32),     # plane kernel
    (6, inputs.BC_PERIODIC, inputs.GEOM_AFFINE, (2, 3, 14), 16),     # plane kernel, 12 slabs of 1-2 layers, periodic plane 0 last
    (7, inputs.BC_PERIODIC, inputs.GEOM_AFFINE, (2, 2, 5), 10),      # line kernel, vector tail
    (4, inputs.BC_DIRICHLET, inputs.GEOM_AFFINE, (3, 3, 2), 8),      # two slabs
    (8, inputs.BC_PERIODIC, inputs.GEOM_QPOINT, (2, 2, 4), 6),       # full-metric kernel
    (5, inputs.BC_DIRICHLET, inputs.GEOM_QPOINT, (2, 3, 6), 8),
])
def test_apply_host_z_slab_pipeline(env, p, bc, geom, nc, nvec):
    """fe_mf_apply_host pipelined over z-slabs (contiguous copies; chunk k's kernel is an item range of the persistent
    kernel and starts when its planes have landed; its planes of Y leave when it is done): variant 23 forces it on
    small meshes.  Repeated, from a NaN-filled host output; the column-chunk path (variant 22) must agree."""
    torch, orc, binding = env
    w = inputs.Workload(f"host_slabs_p{p}", p, nc, bc, geom, 0.8, (0.0, 0.0, 0.0), (1.0, 1.5, 2.0), nvec, 7700 + p,
                        perturb=0.1 if geom == inputs.GEOM_QPOINT else 0.0)
    X = inputs.multivector(w.seed, w.ndof, nvec)
    Yo = orc.Operator(oracle_mesh(orc, w), w.sigma).apply(X)
    op = binding.FeMf.from_workload(w)
    Xh = torch.from_numpy(X).contiguous().pin_memory()
    Yh = torch.empty_like(Xh).pin_memory()
    op.set_variant(23)
    for rep in range(20):
        Yh.fill_(float("nan"))
        op.apply_host(Xh, Yh, nvec)
        assert relerr(Yh.numpy(), Yo) <= TOL
    assert op.last_launch_count() == min(nc[2], 12)
    op.set_variant(22)
    Yh.fill_(float("nan"))
    op.apply_host(Xh, Yh, nvec)
    assert relerr(Yh.numpy(), Yo) <= TOL
