"""GPU parity of Eq. 17 in full: V = sum_t P^T C^T (sum_e Q^T A Q) C P U -- the constraint matrices of
include/fe_constraints.h inside the decomposed apply (dd.SlabGroup.apply(constraints=...), all tasks on one device) against
the oracle's dd_constrained_apply and against C^T A C of the undecomposed mesh, <= 1e-12.
(The file name keeps these tests, written after GPU access had closed, behind the rest of the suite.)"""
import numpy as np
import pytest

from paper_2208_07129_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = 1e-12


def plane_sets(nd, seed):
    """Closed sets in global node indices, every set inside one node plane: per plane a master-less set of two nodes and
    a set with three masters and two slaves."""
    rng = np.random.default_rng(seed)
    plane = nd[0] * nd[1]
    sets = []
    for iz in range(nd[2]):
        nodes = iz * plane + rng.permutation(plane)
        sets.append(([], nodes[:2], np.zeros((2, 0)), None))
        sets.append((nodes[2:5], nodes[5:7], rng.uniform(-1, 1, (2, 3)), None))
    return sets


CASES = [
    (6, inputs.BC_PERIODIC, inputs.GEOM_AFFINE, (2, 2, 4), 16),
    (4, inputs.BC_DIRICHLET, inputs.GEOM_AFFINE, (3, 2, 4), 8),
    (3, inputs.BC_PERIODIC, inputs.GEOM_QPOINT, (2, 2, 4), 4),
]


@pytest.mark.parametrize("p,bc,geom,nc,nvec", CASES)
@pytest.mark.parametrize("nslabs", [1, 2, 4])
def test_constraints_inside_the_decomposed_apply(p, bc, geom, nc, nvec, nslabs):
    import torch
    from oracle import constraints_oracle as co
    from oracle import dd_oracle as ddo
    from oracle import fe_oracle as orc
    from paper_2208_07129_b200 import dd
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    w = inputs.Workload(f"ddk_p{p}", p, nc, bc, geom, 0.8, (0.0, 0.0, 0.0), (1.0, 1.5, 2.0), nvec, 9900 + p,
                        perturb=0.1 if geom == inputs.GEOM_QPOINT else 0.0)
    bcs = "periodic" if bc == inputs.BC_PERIODIC else "dirichlet"
    op = orc.Operator(orc.Mesh(w.ncells, w.p, bcs, w.box_lo, w.box_hi, vertices=inputs.workload_vertices(w)), w.sigma)
    sets = plane_sets(w.nd, 40 + p)
    S = [co.ConstraintSet(m, s, W, b) for (m, s, W, b) in sets]
    X = inputs.multivector(w.seed, w.ndof, nvec)
    Yo = ddo.dd_constrained_apply(op, X, nslabs, S)
    Yg = co.distribute_transpose(S, op.apply(co.distribute(S, X, homogeneous=True)))
    assert np.abs(Yo - Yg).max() <= 1e-13 * np.abs(Yg).max()
    grp = dd.SlabGroup(w, nslabs)
    cons = [dd.device_constraints(sets, pl) for pl in grp.plans]
    Xd = torch.from_numpy(X.reshape(-1)).cuda()
    U = grp.scatter(Xd, nvec)
    V = [torch.full_like(u, float("nan")) for u in U]
    grp.apply(U, V, nvec, constraints=cons)
    out = grp.gather(V, nvec, torch.full_like(Xd, float("nan")))
    torch.cuda.synchronize()
    got = out.cpu().numpy().reshape(Yo.shape)
    assert np.abs(got - Yo).max() <= TOL * np.abs(Yo).max()
    for I in S:                                              # slave rows of the result are zero (zero columns of C)
        assert np.all(got[I.slaves] == 0.0)
