"""world_size-2 and -3 gloo tests of the decomposed apply's host logic (paper_2208_07129_b200/
dd.py): slab bookkeeping, neighbour ranks, the order of the point-to-point messages of PAPER.md:742-790 (Alg. 5) and
the halo add.  The two DEVICE calls of a task (local apply, halo add) are replaced by the CPU oracle / a tensor add
-- injected through dd.LocalOps -- so that the message pattern runs here without a GPU; the same dd_apply_rank drives
NCCL messages between GPUs.  The single-process form (dd.SlabGroup) is exercised with the same stand-ins."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import dd_oracle as ddo
from oracle import fe_oracle as orc
from paper_2208_07129_b200 import dd, inputs


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _workload(bc):
    return inputs.Workload("dd_host", 3, (2, 2, 5), bc, inputs.GEOM_AFFINE, 0.7, (0.0, 0.0, 0.0), (1.0, 1.5, 2.5), 3, 4321)


def _oracle_ops(w, plan):
    """Stand-ins for fe_mf_apply on a slab context and fe_mf_halo_add (host logic tests only)."""
    bc = "periodic" if w.bc == inputs.BC_PERIODIC else "dirichlet"
    op = orc.Operator(orc.Mesh(w.ncells, w.p, bc, w.box_lo, w.box_hi), w.sigma)

    def apply(U, V, nvec):
        V.copy_(torch.from_numpy(ddo.slab_apply(op, plan.z0, plan.z1, U.numpy().reshape(-1, nvec).copy()).reshape(-1)))

    def unpack_f32(dst, src, add):
        return dst.add_(src.double()) if add else dst.copy_(src.double())

    def axpby(Z, W, beta, gamma):
        return Z.copy_(gamma * W) if beta == 0.0 else Z.mul_(beta).add_(W, alpha=gamma)

    return dd.LocalOps(apply=apply, halo_add=lambda dst, src: dst.add_(src),
                       pack_f32=lambda dst, src: dst.copy_(src.to(torch.float32)), unpack_f32=unpack_f32, axpby=axpby)


def _worker_batches(rank, world, port, bc, q, fp32=False):
    """Alg. 5: three batches of the multivector, exchange of batch i+1 / halo add of batch i-1 in flight during batch i."""
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = _workload(bc)
        nvec, nb = w.nvec, 3
        plan = dd.make_plan(w.ncells, w.p, bc == inputs.BC_PERIODIC, world, rank)
        pe = plan.plane_nodes * nvec
        first = plan.z0 * plan.p
        Us, Vs = [], []
        for b in range(nb):
            X = inputs.multivector(w.seed + 10 * b, w.ndof, nvec)
            U = torch.full((plan.nplanes * pe,), float("nan"), dtype=torch.float64)
            U[:plan.n_owned_planes * pe] = torch.from_numpy(X.reshape(-1)[first * pe:(first + plan.n_owned_planes) * pe].copy())
            Us.append(U); Vs.append(torch.full_like(U, float("nan")))
        dd.dd_apply_rank_batches(plan, _oracle_ops(w, plan), Us, Vs, nvec, dist, fp32_payload=fp32)
        q.put((rank, plan.z0, plan.n_owned_planes, [V[:plan.n_owned_planes * pe].numpy().copy() for V in Vs]))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("bc,fp32", [(inputs.BC_PERIODIC, False), (inputs.BC_DIRICHLET, False), (inputs.BC_PERIODIC, True)])
@pytest.mark.parametrize("world", [2, 3])
def test_decomposed_apply_batches_overlap_over_gloo(bc, fp32, world):
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker_batches, args=(r, world, port, bc, q, fp32)) for r in range(world)]
    for p in procs: p.start()
    res = sorted((q.get(timeout=240) for _ in range(world)), key=lambda r: r[0])
    for p in procs: p.join(timeout=60)
    assert all(p.exitcode == 0 for p in procs)
    w = _workload(bc)
    bcs = "periodic" if bc == inputs.BC_PERIODIC else "dirichlet"
    op = orc.Operator(orc.Mesh(w.ncells, w.p, bcs, w.box_lo, w.box_hi), w.sigma)
    plane = w.nd[0] * w.nd[1] * w.nvec
    for b in range(3):
        Xb = inputs.multivector(w.seed + 10 * b, w.ndof, w.nvec)
        Y = ddo.dd_apply(op, Xb, world, fp32_payload=True) if fp32 else op.apply(Xb)
        for rank, z0, nown, Vs in res:
            ref = Y.reshape(-1)[z0 * w.p * plane:(z0 * w.p + nown) * plane]
            assert np.abs(Vs[b] - ref).max() <= 1e-13 * np.abs(Y).max(), (b, rank)


def _worker(rank, world, port, bc, q, fp32=False):
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = _workload(bc)
        nvec = w.nvec
        plan = dd.make_plan(w.ncells, w.p, bc == inputs.BC_PERIODIC, world, rank)
        X = inputs.multivector(w.seed, w.ndof, nvec)                       # every rank can generate the global block
        pe = plan.plane_nodes * nvec
        U = torch.full((plan.nplanes * pe,), float("nan"), dtype=torch.float64)
        first = plan.z0 * plan.p
        U[:plan.n_owned_planes * pe] = torch.from_numpy(X.reshape(-1)[first * pe:(first + plan.n_owned_planes) * pe].copy())
        V = torch.full_like(U, float("nan"))
        dd.dd_apply_rank(plan, _oracle_ops(w, plan), U, V, nvec, dist, fp32_payload=fp32)
        q.put((rank, plan.z0, plan.z1, plan.n_owned_planes, V[:plan.n_owned_planes * pe].numpy().copy()))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("bc,fp32", [(inputs.BC_PERIODIC, False), (inputs.BC_DIRICHLET, False), (inputs.BC_DIRICHLET, True),
                                     (inputs.BC_PERIODIC, True)])
@pytest.mark.parametrize("world", [2, 3])
def test_decomposed_apply_over_gloo(bc, fp32, world):
    """fp32: the planes travel as FP32; the result is then the oracle's fp32_payload result (the same
    roundings at the same places), which differs from the exact apply at the FP32 level."""
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, bc, q, fp32)) for r in range(world)]
    for p in procs: p.start()
    res = sorted((q.get(timeout=180) for _ in range(world)), key=lambda r: r[0])
    for p in procs: p.join(timeout=60)
    assert all(p.exitcode == 0 for p in procs)
    w = _workload(bc)
    bcs = "periodic" if bc == inputs.BC_PERIODIC else "dirichlet"
    op = orc.Operator(orc.Mesh(w.ncells, w.p, bcs, w.box_lo, w.box_hi), w.sigma)
    X = inputs.multivector(w.seed, w.ndof, w.nvec)
    Y = op.apply(X)
    if fp32:
        Yexact, Y = Y, ddo.dd_apply(op, X, world, fp32_payload=True)
        assert np.abs(Y - Yexact).max() > 1e-10 * np.abs(Y).max()
    plane = w.nd[0] * w.nd[1] * w.nvec
    covered = 0
    for rank, z0, z1, nown, Vown in res:
        first = z0 * w.p
        ref = Y.reshape(-1)[first * plane:(first + nown) * plane]
        assert np.abs(Vown - ref).max() <= 1e-13 * np.abs(Y).max(), (rank, z0, z1)
        covered += nown
    assert covered == w.nd[2]                                              # the owned planes partition the mesh


@pytest.mark.parametrize("fp32", [False, True])
@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_DIRICHLET])
@pytest.mark.parametrize("nslabs", [1, 2, 4, 5])
def test_slab_group_single_process(bc, nslabs, fp32):
    """dd.SlabGroup (all tasks in one process: the single-GPU form) with the oracle stand-ins: scatter, exchange,
    local applies, halo adds, gather = the single-domain apply."""
    w = _workload(bc)
    nvec = w.nvec
    grp = dd.SlabGroup(w, nslabs, make_ops=_oracle_ops)
    X = inputs.multivector(w.seed, w.ndof, nvec)
    Xt = torch.from_numpy(X.reshape(-1).copy())
    U = grp.scatter(Xt, nvec)
    V = [torch.full_like(u, float("nan")) for u in U]
    grp.apply(U, V, nvec, fp32_payload=fp32)
    out = grp.gather(V, nvec, torch.full_like(Xt, float("nan")))
    bcs = "periodic" if bc == inputs.BC_PERIODIC else "dirichlet"
    op = orc.Operator(orc.Mesh(w.ncells, w.p, bcs, w.box_lo, w.box_hi), w.sigma)
    Y = ddo.dd_apply(op, X, nslabs, fp32_payload=True) if fp32 else op.apply(X)
    assert np.abs(out.numpy().reshape(Y.shape) - Y).max() <= 1e-13 * np.abs(Y).max()


def test_plan_bookkeeping():
    """Neighbours, cut-plane masks and sizes of every task."""
    for periodic in (True, False):
        for ns in (1, 2, 3):
            plans = [dd.make_plan((2, 3, 6), 4, periodic, ns, t) for t in range(ns)]
            assert sum(pl.n_owned_planes for pl in plans) == (6 * 4 if periodic else 6 * 4 + 1)
            for t, pl in enumerate(plans):
                assert pl.nplanes == (pl.z1 - pl.z0) * 4 + 1
                if periodic:
                    assert pl.z_open == 3 and pl.up == (t + 1) % ns and pl.down == (t - 1) % ns and pl.has_ghost
                else:
                    assert pl.z_open == ((1 if t > 0 else 0) | (2 if t < ns - 1 else 0))
                    assert pl.up == (t + 1 if t < ns - 1 else None) and pl.down == (t - 1 if t > 0 else None)
                    assert pl.has_ghost == (t < ns - 1)
    assert dd.slab_layers(7, 3) == [(0, 3), (3, 5), (5, 7)]


# ---- the Chebyshev filter on a decomposed mesh ----------------------------------------------------------------------

def _filter_interval(w):
    bcs = "periodic" if w.bc == inputs.BC_PERIODIC else "dirichlet"
    op = orc.Operator(orc.Mesh(w.ncells, w.p, bcs, w.box_lo, w.box_hi), w.sigma)
    b = orc.lanczos_upper_bound(op.apply, inputs.uniform_pm1(w.seed + 1, 0, w.ndof), 10)
    return op, 0.4 * b, b, 0.0


def _worker_cheb(rank, world, port, bc, m, fp32, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = _workload(bc)
        nvec = w.nvec
        _, a, b, a0 = _filter_interval(w)
        plan = dd.make_plan(w.ncells, w.p, bc == inputs.BC_PERIODIC, world, rank)
        pe = plan.plane_nodes * nvec
        first = plan.z0 * plan.p
        Xg = inputs.multivector(w.seed, w.ndof, nvec)
        X = torch.full((plan.nplanes * pe,), float("nan"), dtype=torch.float64)
        X[:plan.n_owned_planes * pe] = torch.from_numpy(Xg.reshape(-1)[first * pe:(first + plan.n_owned_planes) * pe].copy())
        Y = torch.full_like(X, float("nan")); V = torch.full_like(X, float("nan"))
        res, prev = dd.dd_cheb_filter_rank(plan, _oracle_ops(w, plan), X, Y, V, nvec, m, a, b, a0, dist, fp32_payload=fp32)
        assert {res.data_ptr(), prev.data_ptr()} == {X.data_ptr(), Y.data_ptr()}
        q.put((rank, plan.z0, plan.n_owned_planes, res[:plan.n_owned_planes * pe].numpy().copy()))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("bc,m,fp32", [(inputs.BC_PERIODIC, 4, False), (inputs.BC_DIRICHLET, 5, False), (inputs.BC_PERIODIC, 3, True)])
def test_decomposed_chebyshev_filter_over_gloo(bc, m, fp32):
    """world 2: Alg. 6 with every product through the point-to-point exchange; odd and even m (the result ends in either
    buffer); the FP32 payload against the oracle that rounds the same planes in every step."""
    world = 2
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker_cheb, args=(r, world, port, bc, m, fp32, q)) for r in range(world)]
    for p in procs: p.start()
    res = sorted((q.get(timeout=300) for _ in range(world)), key=lambda r: r[0])
    for p in procs: p.join(timeout=60)
    assert all(p.exitcode == 0 for p in procs)
    w = _workload(bc)
    op, a, b, a0 = _filter_interval(w)
    X = inputs.multivector(w.seed, w.ndof, w.nvec)
    Y = ddo.dd_chebyshev_filter(op, X, world, m, a, b, a0, fp32_payload=fp32)
    if not fp32:
        assert np.abs(Y - orc.chebyshev_filter(op.apply, X, m, a, b, a0)).max() <= 1e-12 * np.abs(Y).max()
    plane = w.nd[0] * w.nd[1] * w.nvec
    for rank, z0, nown, Yown in res:
        ref = Y.reshape(-1)[z0 * w.p * plane:(z0 * w.p + nown) * plane]
        assert np.abs(Yown - ref).max() <= 1e-12 * np.abs(Y).max(), rank


@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_DIRICHLET])
@pytest.mark.parametrize("nslabs,m", [(1, 3), (3, 4), (5, 6)])
def test_slab_group_chebyshev_filter_single_process(bc, nslabs, m):
    w = _workload(bc)
    nvec = w.nvec
    op, a, b, a0 = _filter_interval(w)
    grp = dd.SlabGroup(w, nslabs, make_ops=_oracle_ops)
    X = inputs.multivector(w.seed, w.ndof, nvec)
    Xt = torch.from_numpy(X.reshape(-1).copy())
    Xl = grp.scatter(Xt, nvec)
    Yl = [torch.full_like(u, float("nan")) for u in Xl]
    Vl = [torch.full_like(u, float("nan")) for u in Xl]
    res, prev = grp.cheb_filter(Xl, Yl, Vl, nvec, m, a, b, a0)
    out = grp.gather(res, nvec, torch.full_like(Xt, float("nan")))
    Y = orc.chebyshev_filter(op.apply, X, m, a, b, a0)
    assert np.abs(out.numpy().reshape(Y.shape) - Y).max() <= 1e-12 * np.abs(Y).max()
    # the second return value is iterate m - 1 (fe_cheb_filter's contract for X)
    outp = grp.gather(prev, nvec, torch.full_like(Xt, float("nan")))
    Yp = orc.chebyshev_filter(op.apply, X, m - 1, a, b, a0) if m > 1 else X
    assert np.abs(outp.numpy().reshape(Y.shape) - Yp).max() <= 1e-12 * np.abs(Yp).max()


def test_cheb_steps_are_algorithm_6():
    """The scalar recurrence against the oracle's filter on a 1 x 1 'matrix' (apply = multiplication by lambda)."""
    a, b, a0, lam = 1.0, 3.0, 0.2, 0.7
    for m in (1, 2, 5, 8):
        x, y = 1.0, None
        for st in dd.cheb_steps(m, a, b, a0):
            if st[0] == "first":
                y = st[1] * lam * x + st[2] * x
            else:
                x, y = y, st[1] * lam * y + st[2] * x + st[3] * y
        ref = orc.chebyshev_filter(lambda v: lam * v, np.array([[1.0]]), m, a, b, a0)[0, 0]
        assert abs(y - ref) <= 1e-14 * abs(ref)
    with pytest.raises(ValueError):
        list(dd.cheb_steps(3, 2.0, 1.0, 0.0))


# ---- Eq. 17 in full: constraints inside the decomposed apply --------------------------------------------------------

class _OracleConstraints:
    """Stand-in for constraints.Constraints (host logic tests only): the oracle's C, C^T on the local sets."""

    def __init__(self, local_sets):
        from oracle import constraints_oracle as co
        self.co, self.sets = co, [co.ConstraintSet(m, s, W, b) for (m, s, W, b) in local_sets]

    def distribute(self, U, nvec, homogeneous=False):
        U.copy_(torch.from_numpy(self.co.distribute(self.sets, U.numpy().reshape(-1, nvec), homogeneous=homogeneous).reshape(-1)))

    def distribute_transpose(self, V, nvec):
        V.copy_(torch.from_numpy(self.co.distribute_transpose(self.sets, V.numpy().reshape(-1, nvec)).reshape(-1)))


def _plane_sets(w, seed=17):
    """Closed sets in global node indices, every set inside one node plane (tuples as constraints.Constraints takes them)."""
    rng = np.random.default_rng(seed)
    plane = w.nd[0] * w.nd[1]
    sets = []
    for iz in range(w.nd[2]):
        nodes = iz * plane + rng.permutation(plane)
        sets.append(([], nodes[:2], np.zeros((2, 0)), None))
        sets.append((nodes[2:5], nodes[5:7], rng.uniform(-1, 1, (2, 3)), None))
    return sets


def _constrained_reference(w, sets, X):
    from oracle import constraints_oracle as co
    bcs = "periodic" if w.bc == inputs.BC_PERIODIC else "dirichlet"
    op = orc.Operator(orc.Mesh(w.ncells, w.p, bcs, w.box_lo, w.box_hi), w.sigma)
    S = [co.ConstraintSet(m, s, W, b) for (m, s, W, b) in sets]
    return co.distribute_transpose(S, op.apply(co.distribute(S, X, homogeneous=True)))


def _worker_constrained(rank, world, port, bc, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = _workload(bc)
        nvec = w.nvec
        plan = dd.make_plan(w.ncells, w.p, bc == inputs.BC_PERIODIC, world, rank)
        cons = _OracleConstraints(dd.restrict_sets(_plane_sets(w), plan))
        X = inputs.multivector(w.seed, w.ndof, nvec)
        pe = plan.plane_nodes * nvec
        first = plan.z0 * plan.p
        U = torch.full((plan.nplanes * pe,), float("nan"), dtype=torch.float64)
        U[:plan.n_owned_planes * pe] = torch.from_numpy(X.reshape(-1)[first * pe:(first + plan.n_owned_planes) * pe].copy())
        V = torch.full_like(U, float("nan"))
        dd.dd_apply_rank(plan, _oracle_ops(w, plan), U, V, nvec, dist, constraints=cons)
        q.put((rank, plan.z0, plan.n_owned_planes, V[:plan.n_owned_planes * pe].numpy().copy()))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_DIRICHLET])
def test_constrained_decomposed_apply_over_gloo(bc):
    world = 2
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker_constrained, args=(r, world, port, bc, q)) for r in range(world)]
    for p in procs: p.start()
    res = sorted((q.get(timeout=240) for _ in range(world)), key=lambda r: r[0])
    for p in procs: p.join(timeout=60)
    assert all(p.exitcode == 0 for p in procs)
    w = _workload(bc)
    X = inputs.multivector(w.seed, w.ndof, w.nvec)
    Y = _constrained_reference(w, _plane_sets(w), X)
    plane = w.nd[0] * w.nd[1] * w.nvec
    for rank, z0, nown, Vown in res:
        ref = Y.reshape(-1)[z0 * w.p * plane:(z0 * w.p + nown) * plane]
        assert np.abs(Vown - ref).max() <= 1e-13 * np.abs(Y).max(), rank


@pytest.mark.parametrize("bc", [inputs.BC_PERIODIC, inputs.BC_DIRICHLET])
@pytest.mark.parametrize("nslabs", [1, 3, 5])
def test_slab_group_constrained_apply_single_process(bc, nslabs):
    """nslabs = 1 on the periodic mesh: the task holds plane 0 twice and gets the sets of that plane twice."""
    w = _workload(bc)
    nvec = w.nvec
    sets = _plane_sets(w)
    grp = dd.SlabGroup(w, nslabs, make_ops=_oracle_ops)
    cons = [_OracleConstraints(dd.restrict_sets(sets, pl)) for pl in grp.plans]
    X = inputs.multivector(w.seed, w.ndof, nvec)
    Xt = torch.from_numpy(X.reshape(-1).copy())
    U = grp.scatter(Xt, nvec)
    V = [torch.full_like(u, float("nan")) for u in U]
    grp.apply(U, V, nvec, constraints=cons)
    out = grp.gather(V, nvec, torch.full_like(Xt, float("nan")))
    Y = _constrained_reference(w, sets, X)
    assert np.abs(out.numpy().reshape(Y.shape) - Y).max() <= 1e-13 * np.abs(Y).max()


def test_restrict_sets_bookkeeping():
    w = _workload(inputs.BC_DIRICHLET)                      # (2, 2, 5) cells, p = 3: 16 node planes
    plane = w.nd[0] * w.nd[1]
    plans = [dd.make_plan(w.ncells, w.p, False, 2, t) for t in range(2)]       # layers [0,3) and [3,5): the cut is plane 9
    on_cut = ([9 * plane + 1], [9 * plane + 2], [[1.0]], None)
    below = ([2 * plane], [2 * plane + 3], [[1.0]], None)
    for pl, expect in zip(plans, ([(9, 9), (2, 2)], [(0, 0)])):
        loc = dd.restrict_sets([on_cut, below], pl)
        assert [(m[0] // plane, s[0] // plane) for (m, s, _, _) in loc] == expect       # local plane numbers
    with pytest.raises(ValueError):                          # master above the cut, slave below it
        dd.restrict_sets([([12 * plane], [3 * plane], [[1.0]], None)], plans[0])
    with pytest.raises(ValueError):
        dd.restrict_sets([on_cut], dd.SlabPlan(0, 2, 0, 3, 3, False, plane))   # a hand-made plan without ncz_total
    per = dd.make_plan((2, 2, 5), 3, True, 1, 0)             # a single periodic task: plane 0 twice
    loc = dd.restrict_sets([([1], [2], [[1.0]], None)], per)
    assert [(m[0], s[0]) for (m, s, _, _) in loc] == [(1, 2), (15 * per.plane_nodes + 1, 15 * per.plane_nodes + 2)]
