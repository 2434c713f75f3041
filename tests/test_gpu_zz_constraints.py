"""GPU parity of the constraint matrices C, C^T (include/fe_constraints.h) against
oracle/constraints_oracle.py, and of C^T A C through the fused apply kernels: periodicity and the Dirichlet condition
expressed as constraint sets on an open slab context must reproduce the periodic / Dirichlet operator (oracle and the
library's own periodic / Dirichlet contexts).
(The file name keeps these tests, written after GPU access had closed, behind the rest of the suite.)"""
import numpy as np
import pytest

from paper_2208_07129_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = 1e-12


@pytest.fixture(scope="module")
def env():
    import torch
    from oracle import constraints_oracle as co
    from oracle import fe_oracle as orc
    from paper_2208_07129_b200 import binding, constraints, dd
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    binding.lib()
    return torch, orc, co, binding, constraints, dd


def as_tuples(sets):
    return [(I.masters, I.slaves, I.W, I.b) for I in sets]


def random_sets(co, rng, ndof, nsets):
    """Closed sets: disjoint slaves, masters drawn from the non-slaves and shared between sets; set 0 has no masters."""
    perm = rng.permutation(ndof)
    nslave_total = ndof // 3
    slaves_pool, masters_pool = perm[:nslave_total], perm[nslave_total:]
    cuts = np.sort(rng.choice(np.arange(1, nslave_total), nsets - 1, replace=False))
    sets = []
    for k, sl in enumerate(np.split(slaves_pool, cuts)):
        nm = 0 if k == 0 else int(rng.integers(1, 40))
        ms = rng.choice(masters_pool, nm, replace=False)
        sets.append(co.ConstraintSet(ms, sl, rng.uniform(-1, 1, (len(sl), nm)), rng.uniform(-1, 1, len(sl))))
    return sets


def relerr(a, b):
    return float(np.abs(a - b).max() / max(np.abs(b).max(), 1e-300))


@pytest.mark.parametrize("nvec", [1, 5, 32, 40])
def test_random_closed_sets(env, nvec):
    torch, orc, co, binding, constraints, dd = env
    rng = np.random.default_rng(100 + nvec)
    ndof = 3000
    sets = random_sets(co, rng, ndof, 37)
    cons = constraints.Constraints(ndof, as_tuples(sets))
    assert cons.counts() == (37, sum(len(I.masters) for I in sets), sum(len(I.slaves) for I in sets))
    U = rng.uniform(-1, 1, (ndof, nvec))
    for homogeneous in (False, True):
        Ud = torch.from_numpy(U.reshape(-1).copy()).cuda()
        cons.distribute(Ud, nvec, homogeneous=homogeneous); torch.cuda.synchronize()
        ref = co.distribute(sets, U, homogeneous=homogeneous)
        got = Ud.cpu().numpy().reshape(ref.shape)
        assert relerr(got, ref) <= 1e-13
        free = np.ones(ndof, dtype=bool)
        for I in sets:
            free[I.slaves] = False
        assert np.array_equal(got[free], U[free])                           # only slave rows are written
    Vd = torch.from_numpy(U.reshape(-1).copy()).cuda()
    cons.distribute_transpose(Vd, nvec); torch.cuda.synchronize()
    ref = co.distribute_transpose(sets, U)
    got = Vd.cpu().numpy().reshape(ref.shape)
    assert relerr(got, ref) <= TOL
    for I in sets:
        assert np.all(got[I.slaves] == 0.0)
    cons.close()


@pytest.mark.parametrize("p", [3, 6, 8])
def test_hanging_face_sets(env, p):
    """Two coarse faces, each with its four child faces as four sets that share the face's (p+1)^2 masters (so the
    transpose accumulates into a master from four blocks)."""
    torch, orc, co, binding, constraints, dd = env
    rng = np.random.default_rng(p)
    n2 = (p + 1) ** 2
    ndof, nvec = 2 * 5 * n2 + 50, 12
    perm = rng.permutation(ndof)
    sets, k = [], 0
    for face in range(2):
        masters = perm[k:k + n2]; k += n2
        for child in [(0, 0), (1, 0), (0, 1), (1, 1)]:
            sets.append(co.ConstraintSet(masters, perm[k:k + n2], co.hanging_face_weights(p, child), None)); k += n2
    cons = constraints.Constraints(ndof, as_tuples(sets))
    U = rng.uniform(-1, 1, (ndof, nvec))
    Ud = torch.from_numpy(U.reshape(-1).copy()).cuda()
    cons.distribute(Ud, nvec); torch.cuda.synchronize()
    assert relerr(Ud.cpu().numpy().reshape(U.shape), co.distribute(sets, U)) <= 1e-13
    Vd = torch.from_numpy(U.reshape(-1).copy()).cuda()
    cons.distribute_transpose(Vd, nvec); torch.cuda.synchronize()
    assert relerr(Vd.cpu().numpy().reshape(U.shape), co.distribute_transpose(sets, U)) <= TOL
    # adjointness on the device results themselves: <C U, V> = <U, C^T V>
    V = rng.uniform(-1, 1, (ndof, nvec))
    a = torch.from_numpy(U.reshape(-1).copy()).cuda(); b = torch.from_numpy(V.reshape(-1).copy()).cuda()
    cons.distribute(a, nvec, homogeneous=True); cons.distribute_transpose(b, nvec); torch.cuda.synchronize()
    lhs = float(np.sum(a.cpu().numpy() * V.reshape(-1))); rhs = float(np.sum(U.reshape(-1) * b.cpu().numpy()))
    assert abs(lhs - rhs) <= 1e-11 * max(abs(lhs), 1.0)


@pytest.mark.parametrize("form", ["one_dense_set", "one_set_per_node"])
@pytest.mark.parametrize("p,nc,nvec,geom", [(6, (2, 3, 3), 16, inputs.GEOM_AFFINE), (7, (2, 2, 3), 8, inputs.GEOM_AFFINE),
                                            (4, (3, 2, 3), 4, inputs.GEOM_QPOINT)])
def test_periodicity_as_a_constraint_on_an_open_slab(env, p, nc, nvec, geom, form):
    """C^T A_open C = the periodic operator (Eq. 17 with one task): the whole periodic mesh as one slab context
    (cut planes open: its top plane duplicates plane 0), the duplication expressed as constraint sets."""
    torch, orc, co, binding, constraints, dd = env
    w = inputs.Workload(f"cons_per_p{p}", p, nc, inputs.BC_PERIODIC, geom, 0.8, (0.0, 0.0, 0.0), (1.0, 1.5, 2.0), nvec, 9500 + p,
                        perturb=0.1 if geom == inputs.GEOM_QPOINT else 0.0)
    plan = dd.make_plan(w.ncells, w.p, True, 1, 0)
    _, ctx = dd.device_ops(w, plan)
    plane = plan.plane_nodes
    nloc = plan.nplanes * plane
    assert ctx.ndofs == nloc == w.ndof + plane
    bottom, top = np.arange(plane), np.arange(w.ndof, nloc)
    if form == "one_dense_set":
        sets = [(bottom, top, np.eye(plane), None)]
    else:
        sets = [([m], [s], [[1.0]], None) for m, s in zip(bottom, top)]
    cons = constraints.Constraints(nloc, sets)
    X = inputs.multivector(w.seed, w.ndof, nvec)
    rng = np.random.default_rng(1)
    Xloc = np.vstack([X, rng.uniform(-9, 9, (plane, nvec))])                 # garbage in the slave rows
    Xd = torch.from_numpy(Xloc.reshape(-1).copy()).cuda()
    Yd = torch.full_like(Xd, float("nan"))
    constraints.constrained_apply(ctx, cons, Xd, Yd, nvec); torch.cuda.synchronize()
    got = Yd.cpu().numpy().reshape(-1, nvec)
    Yo = orc.Operator(orc.Mesh(w.ncells, w.p, "periodic", w.box_lo, w.box_hi, vertices=inputs.workload_vertices(w)), w.sigma).apply(X)
    assert relerr(got[:w.ndof], Yo) <= TOL
    assert np.all(got[w.ndof:] == 0.0)
    assert np.array_equal(Xd.cpu().numpy(), Xloc.reshape(-1))                 # X untouched
    Yp = torch.full((w.ndof * nvec,), float("nan"), dtype=torch.float64, device="cuda")
    binding.FeMf.from_workload(w).apply(torch.from_numpy(X.reshape(-1).copy()).cuda(), Yp, nvec); torch.cuda.synchronize()
    assert relerr(got[:w.ndof].reshape(-1), Yp.cpu().numpy()) <= 1e-13


@pytest.mark.parametrize("p,nvec", [(4, 8), (6, 16)])
def test_dirichlet_as_masterless_sets_on_an_open_slab(env, p, nvec):
    """the Dirichlet condition through the same framework with empty master arrays.  The two middle cell
    layers of a taller Dirichlet mesh as a slab context (both z faces cut planes) + master-less sets on its end planes
    = the Dirichlet operator of the two-layer mesh."""
    torch, orc, co, binding, constraints, dd = env
    h = 0.5
    tall = inputs.Workload("cons_dir_tall", p, (2, 3, 4), inputs.BC_DIRICHLET, inputs.GEOM_AFFINE, 0.9, (0.0, 0.0, 0.0),
                           (1.0, 1.2, 4 * h), nvec, 9600 + p)
    short = inputs.Workload("cons_dir_short", p, (2, 3, 2), inputs.BC_DIRICHLET, inputs.GEOM_AFFINE, 0.9, (0.0, 0.0, h),
                            (1.0, 1.2, 3 * h), nvec, 9600 + p)
    plane = (2 * p + 1) * (3 * p + 1)
    plan = dd.SlabPlan(rank=1, nslabs=3, z0=1, z1=3, p=p, periodic=False, plane_nodes=plane)
    assert plan.z_open == 3
    _, ctx = dd.device_ops(tall, plan)
    assert ctx.ndofs == short.ndof
    ends = np.concatenate([np.arange(plane), np.arange(short.ndof - plane, short.ndof)])
    cons = constraints.Constraints(short.ndof, [([], ends, np.zeros((len(ends), 0)), None)])
    X = inputs.multivector(short.seed, short.ndof, nvec)
    Xd = torch.from_numpy(X.reshape(-1).copy()).cuda()
    Yd = torch.full_like(Xd, float("nan"))
    constraints.constrained_apply(ctx, cons, Xd, Yd, nvec); torch.cuda.synchronize()
    Yo = orc.Operator(orc.Mesh(short.ncells, p, "dirichlet", short.box_lo, short.box_hi), short.sigma).apply(X)
    got = Yd.cpu().numpy().reshape(Yo.shape)
    assert relerr(got, Yo) <= TOL
    assert np.all(got[ends] == 0.0)
    Ys = torch.full_like(Xd, float("nan"))
    binding.FeMf.from_workload(short).apply(Xd, Ys, nvec); torch.cuda.synchronize()
    assert relerr(got.reshape(-1), Ys.cpu().numpy()) <= 1e-13


def test_constraints_argument_errors_on_the_device(env):
    torch, orc, co, binding, constraints, dd = env
    cons = constraints.Constraints(10, [([1], [2], [[0.5]], [0.25])])
    L = constraints.lib()
    U = torch.arange(10, dtype=torch.float64, device="cuda")
    assert L.fe_constraints_distribute(cons._h, None, 1, 0, None) == binding.FE_MF_EINVAL
    assert b"null" in L.fe_constraints_last_error(cons._h)
    assert L.fe_constraints_distribute(cons._h, U.data_ptr(), 0, 0, None) == binding.FE_MF_EINVAL
    cons.distribute(U, 1); torch.cuda.synchronize()
    assert U[2].item() == 0.5 * 1.0 + 0.25
    empty = constraints.Constraints(10, [])
    empty.distribute(U, 1); empty.distribute_transpose(U, 1); torch.cuda.synchronize()
    assert U[2].item() == 0.75 and empty.counts() == (0, 0, 0)
