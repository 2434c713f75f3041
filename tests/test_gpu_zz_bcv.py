"""GPU parity of fe_mf_apply_bcv (the paper's Batched Contiguous Vector layout, Fig. 1) against the
oracle apply, the layout conversion being the oracle's (fe_oracle.to_bcv / from_bcv), <= 1e-12.
(The file name keeps these tests, written after GPU access had closed, behind the rest of the suite.)"""
import numpy as np
import pytest

from paper_2208_07129_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = 1e-12

CASES = [
    # p, bc, geom, cells, nvec, b
    (6, inputs.BC_PERIODIC, inputs.GEOM_AFFINE, (2, 3, 2), 40, 16),     # plane kernel per batch, ragged last batch (8)
    (7, inputs.BC_DIRICHLET, inputs.GEOM_AFFINE, (2, 2, 3), 24, 8),     # line kernel, three full batches
    (8, inputs.BC_PERIODIC, inputs.GEOM_QPOINT, (2, 2, 2), 10, 4),      # full metric, last batch of 2
    (3, inputs.BC_DIRICHLET, inputs.GEOM_AFFINE, (3, 2, 2), 7, 3),      # odd widths: loads / atomics kernels; offsets only 8-byte aligned
    (4, inputs.BC_PERIODIC, inputs.GEOM_AFFINE, (2, 2, 2), 6, 8),       # b >= nvec: the plain layout
    (2, inputs.BC_PERIODIC, inputs.GEOM_AFFINE, (3, 3, 3), 5, 1),       # one vector per batch
]


@pytest.mark.parametrize("p,bc,geom,nc,nvec,b", CASES)
def test_apply_bcv_matches_the_oracle(p, bc, geom, nc, nvec, b):
    import torch
    from oracle import fe_oracle as orc
    from paper_2208_07129_b200 import binding
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    w = inputs.Workload(f"bcv_p{p}", p, nc, bc, geom, 0.8, (0.0, 0.0, 0.0), (1.0, 1.5, 2.0), nvec, 9700 + p,
                        perturb=0.1 if geom == inputs.GEOM_QPOINT else 0.0)
    bcs = "periodic" if bc == inputs.BC_PERIODIC else "dirichlet"
    op_o = orc.Operator(orc.Mesh(w.ncells, w.p, bcs, w.box_lo, w.box_hi, vertices=inputs.workload_vertices(w)), w.sigma)
    X = inputs.multivector(w.seed, w.ndof, nvec)
    Yo = op_o.apply(X)
    op = binding.FeMf.from_workload(w)
    Xd = torch.from_numpy(orc.to_bcv(X, b)).cuda()
    Yd = torch.full_like(Xd, float("nan"))
    op.apply_bcv(Xd, Yd, b, nvec); torch.cuda.synchronize()
    got = orc.from_bcv(Yd.cpu().numpy(), w.ndof, nvec, b)
    assert float(np.abs(got - Yo).max() / np.abs(Yo).max()) <= TOL
    assert op.last_launch_count() >= -(-nvec // b)                        # at least one kernel per batch
    with pytest.raises(binding.FeMfError) as e:
        op.apply_bcv(Xd, Xd, b, nvec)
    assert e.value.code == binding.FE_MF_EINVAL
