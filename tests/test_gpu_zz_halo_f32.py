"""GPU parity of the FP32 boundary payload ("the boundary data communicated is
recast as FP32 floats"): fe_mf_halo_pack_f32 / fe_mf_halo_unpack_f32 bit for bit against numpy's IEEE conversions, and the
decomposed apply with the payload (dd.SlabGroup, all tasks on one device) against the oracle that rounds the same
planes at the same places (oracle/dd_oracle.py: dd_apply(fp32_payload=True)), <= 1e-12.
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


def special_values():
    """Doubles that sit on the decision points of the FP64 -> FP32 rounding."""
    e = 2.0 ** -24
    return np.array([0.0, -0.0, 1.0, 1.0 + e, 1.0 + e + 2.0 ** -50, 1.0 + 3 * e, 1.0 - e / 2, -1.0 - e,        # ties go to even
                     3.4028234663852886e38, 3.4028235677973366e38, -3.5e38, 1e39,                                # FLT_MAX, overflow
                     1.1754943508222875e-38, 1e-40, 1.401298464324817e-45, 0.7e-45, 0.70064923216240854e-45,     # subnormals
                     1e-300, -1e-300, np.pi, -np.e, 123456789.123456789], dtype=np.float64)


@pytest.mark.parametrize("count,offset", [(1, 0), (255, 0), (4097, 1), (1 << 20, 3)])
def test_pack_and_unpack_are_the_ieee_conversions_bit_for_bit(env, count, offset):
    torch, orc, ddo, binding, dd = env
    rng = np.random.default_rng(count)
    src = rng.uniform(-1, 1, count) * 10.0 ** rng.integers(-30, 30, count)
    sp = special_values()
    src[:min(count, len(sp))] = sp[:min(count, len(sp))]
    with np.errstate(over="ignore"):
        ref32 = src.astype(np.float32)
    # views offset by `offset` elements: pointers aligned to 8 (double) / 4 (float) bytes only
    s_all = torch.zeros(count + offset, dtype=torch.float64, device="cuda")
    d_all = torch.full((count + offset + 1,), 7.0, dtype=torch.float32, device="cuda")
    s_all[offset:].copy_(torch.from_numpy(src))
    binding.halo_pack_f32(d_all[offset:offset + count], s_all[offset:])
    torch.cuda.synchronize()
    got = d_all.cpu().numpy()
    assert np.array_equal(got[offset:offset + count].view(np.uint32), ref32.view(np.uint32))
    assert np.all(got[:offset] == 7.0) and got[offset + count] == 7.0                   # nothing written outside
    # unpack, overwrite
    back = torch.full((count + offset + 1,), -3.0, dtype=torch.float64, device="cuda")
    binding.halo_unpack_f32(back[offset:offset + count], d_all[offset:offset + count], add=False)
    torch.cuda.synchronize()
    b = back.cpu().numpy()
    assert np.array_equal(b[offset:offset + count].view(np.uint64), ref32.astype(np.float64).view(np.uint64))
    assert np.all(b[:offset] == -3.0) and b[offset + count] == -3.0
    # unpack, add (finite values only: inf + finite is inf on both sides, but keep the comparison simple)
    fin = np.isfinite(ref32)
    base = rng.uniform(-1, 1, count)
    acc = torch.from_numpy(base.copy()).cuda()
    binding.halo_unpack_f32(acc, d_all[offset:offset + count].contiguous(), add=True)
    torch.cuda.synchronize()
    want = base + ref32.astype(np.float64)
    assert np.array_equal(acc.cpu().numpy()[fin].view(np.uint64), want[fin].view(np.uint64))


def test_halo_f32_argument_errors(env):
    torch, orc, ddo, binding, dd = env
    L = binding.lib()
    a = torch.zeros(4, dtype=torch.float64, device="cuda"); b = torch.zeros(4, dtype=torch.float32, device="cuda")
    assert L.fe_mf_halo_pack_f32(None, a.data_ptr(), 4, None) == binding.FE_MF_EINVAL
    assert L.fe_mf_halo_pack_f32(b.data_ptr(), a.data_ptr(), -1, None) == binding.FE_MF_EINVAL
    assert L.fe_mf_halo_unpack_f32(a.data_ptr(), b.data_ptr(), 4, 2, None) == binding.FE_MF_EINVAL
    assert L.fe_mf_halo_unpack_f32(a.data_ptr(), None, 4, 0, None) == binding.FE_MF_EINVAL
    assert L.fe_mf_halo_pack_f32(b.data_ptr(), a.data_ptr(), 0, None) == binding.FE_MF_OK


CASES = [
    (6, inputs.BC_PERIODIC, inputs.GEOM_AFFINE, (2, 3, 5), 16),
    (6, inputs.BC_DIRICHLET, inputs.GEOM_AFFINE, (3, 2, 5), 32),
    (7, inputs.BC_PERIODIC, inputs.GEOM_AFFINE, (2, 2, 4), 10),
    (8, inputs.BC_PERIODIC, inputs.GEOM_QPOINT, (2, 2, 4), 6),
    (3, inputs.BC_DIRICHLET, inputs.GEOM_AFFINE, (3, 2, 4), 3),
]


@pytest.mark.parametrize("p,bc,geom,nc,nvec", CASES)
@pytest.mark.parametrize("nslabs", [1, 2, 4])
def test_slab_group_with_fp32_payload_matches_the_oracle(env, p, bc, geom, nc, nvec, nslabs):
    """The same planes are rounded at the same places on both sides, so the tolerance stays 1e-12 although the result
    is 1e-8 away from the exact apply."""
    torch, orc, ddo, binding, dd = env
    w = inputs.Workload(f"ddf_p{p}", p, nc, bc, geom, 0.8, (0.0, 0.0, 0.0), (1.0, 1.5, 2.0), nvec, 9400 + p,
                        perturb=0.1 if geom == inputs.GEOM_QPOINT else 0.0)
    bcs = "periodic" if bc == inputs.BC_PERIODIC else "dirichlet"
    op = orc.Operator(orc.Mesh(w.ncells, w.p, bcs, w.box_lo, w.box_hi, vertices=inputs.workload_vertices(w)), w.sigma)
    X = inputs.multivector(w.seed, w.ndof, nvec)
    Yo = ddo.dd_apply(op, X, nslabs, fp32_payload=True)
    Yexact = op.apply(X)
    grp = dd.SlabGroup(w, nslabs)
    Xd = torch.from_numpy(X.reshape(-1)).cuda()
    U = grp.scatter(Xd, nvec)
    V = [torch.full_like(u, float("nan")) for u in U]
    grp.apply(U, V, nvec, fp32_payload=True)
    out = grp.gather(V, nvec, torch.full_like(Xd, float("nan")))
    torch.cuda.synchronize()
    got = out.cpu().numpy().reshape(Yo.shape)
    scale = np.abs(Yo).max()
    # the inbound rounding of U is amplified by the operator exactly as in the oracle; what is left is summation order --
    # except where a ghost row of V sits within that roundoff of an FP32 rounding boundary: the two sides may then round
    # it to neighbouring floats (chance ~1e-8 per value).  Such an entry is accepted if it is one FP32 ulp (of the largest
    # value) off, and at most two of them.
    err = np.abs(got - Yo)
    bad = err > TOL * scale
    assert bad.sum() <= 2 and np.all(err[bad] <= 2.0 ** -23 * scale)
    dev = np.abs(got - Yexact).max() / scale
    if nslabs == 1:
        assert dev <= TOL                                              # a single task exchanges nothing
    else:
        assert 1e-10 < dev < 1e-5                                      # the payload really was FP32
