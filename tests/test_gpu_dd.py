"""GPU parity of the decomposed apply: slab contexts (fe_mf_create_slab: cut planes open, no
wrap in z) against the oracle's local operator, and the whole exchange (dd.SlabGroup: all tasks on one device, messages
as device copies, halo add by fe_mf_halo_add) against the single-domain oracle, <= 1e-12."""
import numpy as np
import pytest

from paper_2208_07129_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = 1e-12


@pytest.fixture(scope="module")
def env():
    import torch
    from oracle import dd_oracle as ddo
    from oracle import fe_oracle as orc
    from paper_2208_07129_b200 import binding, dd
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    binding.lib()
    return torch, orc, ddo, binding, dd


def oracle_op(orc, w):
    bc = "periodic" if w.bc == inputs.BC_PERIODIC else "dirichlet"
    return orc.Operator(orc.Mesh(w.ncells, w.p, bc, w.box_lo, w.box_hi, vertices=inputs.workload_vertices(w)), w.sigma)


def relerr(a, b):
    return float(np.abs(a - b).max() / np.abs(b).max())


CASES = [
    # p, bc, geom, cells, nvec            kernel the slab contexts run
    (6, inputs.BC_PERIODIC, inputs.GEOM_AFFINE, (2, 3, 5), 16),      # plane
    (6, inputs.BC_DIRICHLET, inputs.GEOM_AFFINE, (3, 2, 5), 32),     # plane, Dirichlet x / y faces and physical z ends
    (7, inputs.BC_PERIODIC, inputs.GEOM_AFFINE, (2, 2, 4), 10),      # line, vector tail
    (4, inputs.BC_DIRICHLET, inputs.GEOM_AFFINE, (3, 3, 4), 8),      # line
    (8, inputs.BC_PERIODIC, inputs.GEOM_QPOINT, (2, 2, 4), 6),       # full metric, per-q-point
    (5, inputs.BC_DIRICHLET, inputs.GEOM_QPOINT, (2, 3, 4), 8),
    (3, inputs.BC_PERIODIC, inputs.GEOM_AFFINE, (3, 2, 4), 3),       # odd nvec: loads / atomics kernels
    (2, inputs.BC_DIRICHLET, inputs.GEOM_AFFINE, (3, 2, 4), 1),      # single vector
]


@pytest.mark.parametrize("p,bc,geom,nc,nvec", CASES)
def test_slab_context_matches_the_oracle_local_operator(env, p, bc, geom, nc, nvec):
    """V^(t) = A^(t) U^(t) of every task of a 2- and a 3-slab decomposition, all local rows (owned and ghost), from
    a local multivector whose ghost plane is filled (P^(t) U)."""
    torch, orc, ddo, binding, dd = env
    w = inputs.Workload(f"dd_p{p}", p, nc, bc, geom, 0.8, (0.0, 0.0, 0.0), (1.0, 1.5, 2.0), nvec, 9100 + p,
                        perturb=0.1 if geom == inputs.GEOM_QPOINT else 0.0)
    op_o = oracle_op(orc, w)
    X = inputs.multivector(w.seed, w.ndof, nvec)
    for nslabs in (2, 3):
        for t in range(nslabs):
            plan = dd.make_plan(w.ncells, w.p, bc == inputs.BC_PERIODIC, nslabs, t)
            rows, _ = ddo.slab_rows(op_o.mesh, plan.z0, plan.z1)
            U = X[rows].copy()
            Vo = ddo.slab_apply(op_o, plan.z0, plan.z1, U)
            _, ctx = dd.device_ops(w, plan)
            assert ctx.ndofs == len(rows)
            Ud = torch.from_numpy(U.reshape(-1)).cuda()
            Vd = torch.full_like(Ud, float("nan"))
            ctx.apply(Ud, Vd, nvec); torch.cuda.synchronize()
            assert relerr(Vd.cpu().numpy().reshape(Vo.shape), Vo) <= TOL, (nslabs, t, ctx.kernel_name(nvec))


@pytest.mark.parametrize("p,bc,geom,nc,nvec", CASES)
@pytest.mark.parametrize("nslabs", [1, 2, 4])
def test_slab_group_matches_single_domain(env, p, bc, geom, nc, nvec, nslabs):
    """scatter -> ghost exchange -> local fused kernels -> halo add -> gather = A X of the undecomposed mesh (oracle and
    the undecomposed GPU context)."""
    torch, orc, ddo, binding, dd = env
    w = inputs.Workload(f"ddg_p{p}", p, nc, bc, geom, 0.8, (0.0, 0.0, 0.0), (1.0, 1.5, 2.0), nvec, 9200 + p,
                        perturb=0.1 if geom == inputs.GEOM_QPOINT else 0.0)
    X = inputs.multivector(w.seed, w.ndof, nvec)
    Yo = oracle_op(orc, w).apply(X)
    grp = dd.SlabGroup(w, nslabs)
    Xd = torch.from_numpy(X.reshape(-1)).cuda()
    U = grp.scatter(Xd, nvec)
    V = [torch.full_like(u, float("nan")) for u in U]
    grp.apply(U, V, nvec)
    out = grp.gather(V, nvec, torch.full_like(Xd, float("nan")))
    torch.cuda.synchronize()
    assert relerr(out.cpu().numpy().reshape(Yo.shape), Yo) <= TOL
    Yd = torch.full_like(Xd, float("nan"))
    binding.FeMf.from_workload(w).apply(Xd, Yd, nvec); torch.cuda.synchronize()
    assert relerr(out.cpu().numpy(), Yd.cpu().numpy()) <= 1e-13


def test_slab_context_refuses_what_needs_the_neighbour(env):
    torch, orc, ddo, binding, dd = env
    w = inputs.Workload("dd_refuse", 4, (2, 2, 4), inputs.BC_PERIODIC, inputs.GEOM_AFFINE, 1.0, (0, 0, 0), (1, 1, 2), 4, 9300)
    _, ctx = dd.device_ops(w, dd.make_plan(w.ncells, w.p, True, 2, 0))
    X = torch.zeros(ctx.ndofs * 4, dtype=torch.float64, device="cuda"); Y = torch.zeros_like(X)
    with pytest.raises(binding.FeMfError) as e:
        ctx.cheb_filter(X, Y, 4, 3, 1.0, 2.0, 0.0)
    assert e.value.code == binding.FE_MF_EUNSUPPORTED
    with pytest.raises(binding.FeMfError):
        ctx.set_mass_scaling(True)
    with pytest.raises(binding.FeMfError):
        binding.FeMf((2, 2, 2), 3, 1.0, inputs.BC_PERIODIC, z_open=1)     # a periodic slab is cut at both faces
