"""GPU parity of the Chebyshev filter on a decomposed mesh (Alg. 6 PAPER.md:941-966 with Alg. 5's
exchange in every step, the paper's multi-GPU eigenproblem runs PAPER.md:1005): dd.SlabGroup.cheb_filter (all tasks on
one device: slab contexts, halo add, fe_mf_axpby on the owned rows) against the oracle's filter, <= 1e-12, and against
fe_cheb_filter of the undecomposed context; fe_mf_axpby against numpy.
(The file name keeps these tests, written after GPU access had closed, behind the rest of the suite.)"""
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


@pytest.mark.parametrize("count,offset", [(1, 0), (1001, 1), (1 << 18, 0)])
def test_axpby_entry_point(env, count, offset):
    torch, orc, ddo, binding, dd = env
    rng = np.random.default_rng(count)
    z, w = rng.uniform(-1, 1, count + offset), rng.uniform(-1, 1, count + offset)
    Z = torch.from_numpy(z.copy()).cuda(); W = torch.from_numpy(w.copy()).cuda()
    binding.axpby(Z[offset:], W[offset:], 0.75, -1.5); torch.cuda.synchronize()
    ref = z.copy(); ref[offset:] = 0.75 * z[offset:] + (-1.5) * w[offset:]
    assert np.abs(Z.cpu().numpy() - ref).max() <= 1e-15
    Zn = torch.full((count + offset,), float("nan"), dtype=torch.float64, device="cuda")
    binding.axpby(Zn[offset:], W[offset:], 0.0, 2.0); torch.cuda.synchronize()      # beta = 0: Z is not read
    got = Zn.cpu().numpy()
    assert np.array_equal(got[offset:], 2.0 * w[offset:]) and np.isnan(got[:offset]).all()
    assert binding.lib().fe_mf_axpby(None, W.data_ptr(), 1.0, 1.0, 4, None) == binding.FE_MF_EINVAL


CASES = [
    # p, bc, geom, cells, nvec, m
    (6, inputs.BC_PERIODIC, inputs.GEOM_AFFINE, (2, 2, 4), 16, 6),      # plane kernel in every slab
    (4, inputs.BC_DIRICHLET, inputs.GEOM_AFFINE, (3, 2, 4), 8, 5),      # line kernel; boundary rows follow the scalar recurrence
    (3, inputs.BC_PERIODIC, inputs.GEOM_QPOINT, (2, 2, 4), 4, 4),       # full metric
]


@pytest.mark.parametrize("p,bc,geom,nc,nvec,m", CASES)
@pytest.mark.parametrize("nslabs,fp32", [(1, False), (2, False), (4, False), (2, True)])
def test_slab_group_chebyshev_filter_matches_the_oracle(env, p, bc, geom, nc, nvec, m, nslabs, fp32):
    torch, orc, ddo, binding, dd = env
    w = inputs.Workload(f"ddc_p{p}", p, nc, bc, geom, 0.8, (0.0, 0.0, 0.0), (1.0, 1.5, 2.0), nvec, 9800 + p,
                        perturb=0.1 if geom == inputs.GEOM_QPOINT else 0.0)
    bcs = "periodic" if bc == inputs.BC_PERIODIC else "dirichlet"
    op = orc.Operator(orc.Mesh(w.ncells, w.p, bcs, w.box_lo, w.box_hi, vertices=inputs.workload_vertices(w)), w.sigma)
    b = orc.lanczos_upper_bound(op.apply, inputs.uniform_pm1(w.seed + 1, 0, w.ndof), 10)
    a, a0 = 0.4 * b, 0.0
    X = inputs.multivector(w.seed, w.ndof, nvec)
    Yo = ddo.dd_chebyshev_filter(op, X, nslabs, m, a, b, a0, fp32_payload=fp32)
    grp = dd.SlabGroup(w, nslabs)
    Xd = torch.from_numpy(X.reshape(-1)).cuda()
    Xl = grp.scatter(Xd, nvec)
    Yl = [torch.full_like(u, float("nan")) for u in Xl]
    Vl = [torch.full_like(u, float("nan")) for u in Xl]
    res, prev = grp.cheb_filter(Xl, Yl, Vl, nvec, m, a, b, a0, fp32_payload=fp32)
    out = grp.gather(res, nvec, torch.full_like(Xd, float("nan")))
    torch.cuda.synchronize()
    got = out.cpu().numpy().reshape(Yo.shape)
    scale = np.abs(Yo).max()
    if fp32:
        # the same planes are rounded at the same places; an entry that sits on an FP32 rounding boundary may round the
        # other way on the two sides, and later steps spread that flip: FP32 level, not the 1e-12 of the exact path
        assert np.abs(got - Yo).max() <= 2.0 ** -20 * scale
        assert np.abs(got - orc.chebyshev_filter(op.apply, X, m, a, b, a0)).max() > 1e-10 * scale
        return
    assert np.abs(got - Yo).max() <= TOL * scale
    # the undecomposed context's filter (scaled recurrence, identity term in the kernel): same polynomial
    ctx = binding.FeMf.from_workload(w)
    Xc = torch.from_numpy(X.reshape(-1)).cuda(); Yc = torch.full_like(Xc, float("nan"))
    ctx.cheb_filter(Xc, Yc, nvec, m, a, b, a0); torch.cuda.synchronize()
    assert np.abs(got.reshape(-1) - Yc.cpu().numpy()).max() <= TOL * scale
