"""Domain-decomposed apply (section 3.2.5 / Alg. 5) on z-slabs.

    V = sum_t P^(t)T A^(t) P^(t) U

One task t per process (one process per GPU, `torch.distributed` for the point-to-point exchange: NCCL between GPUs),
or several tasks in ONE process on one device (`SlabGroup`: the exchange is a device copy), which is how the path is
run and checked on a single B200.  A task owns the cell layers z0 <= ez < z1 and the node planes z0 p <= iz < z1 p; its
local multivector is its owned planes followed by its top plane, the ghost plane, so that both messages
of a task are CONTIGUOUS blocks of the multivector and nothing is packed:

    P^(t):    the owner of the ghost plane (task t+1) sends its first owned plane of U          -> ghost plane of U^(t)
    A^(t):    fe_mf_apply on the slab context (fe_mf_create_slab): the fused kernels, cut planes open
    P^(t)T:   task t sends the ghost plane of V^(t) to task t+1, which ADDS it to its first plane (fe_mf_halo_add)

With `fp32_payload` the plane that crosses a task boundary travels as FP32 ("the boundary data communicated
is recast as FP32 floats"): fe_mf_halo_pack_f32 on the sending side into a message buffer of half the bytes,
fe_mf_halo_unpack_f32 on the receiving side (overwrite for U, add for V); everything a task computes stays FP64.  A
single task exchanges nothing, so nothing is rounded.

dd_cheb_filter_rank / SlabGroup.cheb_filter: the Chebyshev filter (Alg. 6) on a decomposed mesh -- every product by the
exchange above, the three-term update of the owned rows by fe_mf_axpby; the host evaluates the scalar recurrence.

This module is argument marshalling and message ordering only; the arithmetic is in libfe_mf.so.  The local operator
and the halo add are injected (`ops`), so that the message pattern can be exercised without a GPU (tests/
test_dd_gloo.py runs it over gloo with the CPU oracle standing in for the two device calls).
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Callable, List, Optional, Sequence, Tuple


def slab_layers(ncz: int, nslabs: int) -> List[Tuple[int, int]]:
    """Cell layers [z0, z1) of each task: as even as possible, the first ncz % nslabs tasks take one more."""
    if nslabs < 1 or nslabs > ncz:
        raise ValueError("need 1 <= nslabs <= ncz")
    base, rem = divmod(ncz, nslabs)
    out, z = [], 0
    for t in range(nslabs):
        n = base + (1 if t < rem else 0)
        out.append((z, z + n))
        z += n
    return out


@dataclass(frozen=True)
class SlabPlan:
    """Bookkeeping of one task: sizes are in node PLANES of the local multivector (a plane = nd_x nd_y nvec doubles)."""
    rank: int
    nslabs: int
    z0: int
    z1: int
    p: int
    periodic: bool
    plane_nodes: int                 # nd_x * nd_y
    ncz_total: int = 0               # cell layers of the whole mesh (make_plan sets it; needed by restrict_sets only)

    @property
    def nplanes(self) -> int:        # planes of the local multivector (owned + the top plane)
        return (self.z1 - self.z0) * self.p + 1

    @property
    def has_ghost(self) -> bool:     # the top plane belongs to the next task (else it is the Dirichlet boundary plane)
        return self.periodic or self.rank < self.nslabs - 1

    @property
    def up(self) -> Optional[int]:   # owner of the ghost plane
        if not self.has_ghost:
            return None
        return (self.rank + 1) % self.nslabs

    @property
    def down(self) -> Optional[int]:  # the task whose ghost plane is this task's first plane
        if self.periodic:
            return (self.rank - 1) % self.nslabs
        return self.rank - 1 if self.rank > 0 else None

    @property
    def z_open(self) -> int:
        """fe_mf_create_slab's mask: bit 0 / 1 = low / high z face is a cut plane."""
        if self.periodic:
            return 3
        return (1 if self.rank > 0 else 0) | (2 if self.rank < self.nslabs - 1 else 0)

    @property
    def n_owned_planes(self) -> int:
        return self.nplanes - 1 if self.has_ghost else self.nplanes


def make_plan(ncells: Sequence[int], p: int, periodic: bool, nslabs: int, rank: int) -> SlabPlan:
    z0, z1 = slab_layers(ncells[2], nslabs)[rank]
    add = 0 if periodic else 1
    return SlabPlan(rank, nslabs, z0, z1, p, periodic, (ncells[0] * p + add) * (ncells[1] * p + add), ncells[2])


def restrict_sets(sets, plan: SlabPlan):
    """C^(t) of Eq. 17: constraint sets given in GLOBAL node indices -- tuples (masters, slaves, W, b) as
    constraints.Constraints takes them -- restricted to the local rows of task `plan` (host-side index marshalling).  A set
    takes part if one of its slaves is a local row; then all its nodes must be local rows, else ValueError (a set that
    straddles a cut would need masters the task does not hold).  A row on a cut plane is local to two tasks, and a single
    periodic task holds plane 0 twice (first plane and ghost plane): one local set per copy."""
    if plan.ncz_total <= 0:
        raise ValueError("restrict_sets needs a plan from make_plan (ncz_total)")
    ndz = plan.ncz_total * plan.p + (0 if plan.periodic else 1)
    local_planes = {}
    for l in range(plan.nplanes):
        g = plan.z0 * plan.p + l
        local_planes.setdefault(g % ndz if plan.periodic else g, []).append(l)
    pn = plan.plane_nodes
    out = []
    for (masters, slaves, W, b) in sets:
        masters = [int(v) for v in masters]
        slaves = [int(v) for v in slaves]
        if not any(v // pn in local_planes for v in slaves):
            continue
        nodes = masters + slaves
        if not all(v // pn in local_planes for v in nodes):
            raise ValueError("a constraint set straddles a subdomain boundary")
        copies = {len(local_planes[v // pn]) for v in nodes}
        if len(copies) != 1:
            raise ValueError("a constraint set mixes rows the task holds once and rows it holds twice")
        for c in range(copies.pop()):
            loc = lambda v: local_planes[v // pn][c] * pn + v % pn      # noqa: E731
            out.append(([loc(v) for v in masters], [loc(v) for v in slaves], W, b))
    return out


def device_constraints(sets, plan: SlabPlan, device: int = 0):
    """The task's constraint object on the device (include/fe_constraints.h) from sets in global node indices."""
    from . import constraints
    return constraints.Constraints(plan.nplanes * plan.plane_nodes, restrict_sets(sets, plan), device)


def slab_geometry(w, plan: SlabPlan):
    """(ncells, box_lo, box_hi, vertices) of the slab of workload w (paper_2208_07129_b200.inputs.Workload)."""
    from . import inputs
    ncz = w.ncells[2]
    hz = (w.box_hi[2] - w.box_lo[2]) / ncz
    lo = (w.box_lo[0], w.box_lo[1], w.box_lo[2] + hz * plan.z0)
    hi = (w.box_hi[0], w.box_hi[1], w.box_lo[2] + hz * plan.z1)
    verts = inputs.workload_vertices(w)
    if verts is not None:
        verts = verts[plan.z0:plan.z1 + 1].copy()
    return (w.ncells[0], w.ncells[1], plan.z1 - plan.z0), lo, hi, verts


@dataclass
class LocalOps:
    """The device calls of a task: V_loc = A^(t) U_loc; dst += src; for the FP32 payload only, pack_f32(dst32, src64)
    and unpack_f32(dst64, src32, add); for the Chebyshev filter only, axpby(Z, W, beta, gamma): Z <- beta Z + gamma W."""
    apply: Callable
    halo_add: Callable
    pack_f32: Optional[Callable] = None
    unpack_f32: Optional[Callable] = None
    axpby: Optional[Callable] = None


def device_ops(w, plan: SlabPlan, device: int = 0):
    """LocalOps backed by libfe_mf.so (fe_mf_create_slab / fe_mf_apply / fe_mf_halo_add)."""
    from . import binding
    nc, lo, hi, verts = slab_geometry(w, plan)
    op = binding.FeMf(nc, w.p, w.sigma, w.bc, w.geom, lo, hi, verts, device, z_open=plan.z_open)
    return LocalOps(apply=lambda U, V, nvec: op.apply(U, V, nvec), halo_add=binding.halo_add,
                    pack_f32=binding.halo_pack_f32, unpack_f32=binding.halo_unpack_f32, axpby=binding.axpby), op


def _buffers32(like, pe: int, count: int):
    import torch
    return [torch.empty(pe, dtype=torch.float32, device=like.device) for _ in range(count)]


def dd_apply_rank(plan: SlabPlan, ops: LocalOps, U_loc, V_loc, nvec: int, dist, scratch=None, fp32_payload: bool = False,
                  scratch32=None, constraints=None):
    """One task of the decomposed apply with torch.distributed point-to-point messages (dist = torch.distributed).
    U_loc / V_loc: flat tensors of nplanes * plane_nodes * nvec doubles; the ghost plane of U_loc is overwritten.
    `scratch`: one plane, receives the neighbour's ghost plane of V.  fp32_payload: the planes travel as FP32
    (`scratch32`: two float32 planes, the send and the receive buffer).  constraints: the task's C^(t) (an object with
    distribute(U, nvec, homogeneous=True) and distribute_transpose(V, nvec): constraints.Constraints from
    device_constraints) -- Eq. 17 in full, V = sum_t P^T C^T A C P U; the slave rows of U_loc are then overwritten by their
    constrained values."""
    pe = plan.plane_nodes * nvec
    own = plan.n_owned_planes * pe
    if plan.nslabs == 1:                       # a single periodic task is its own neighbour
        if plan.has_ghost:
            U_loc[own:own + pe].copy_(U_loc[:pe])
        if constraints is not None:
            constraints.distribute(U_loc, nvec, homogeneous=True)
        ops.apply(U_loc, V_loc, nvec)
        if constraints is not None:
            constraints.distribute_transpose(V_loc, nvec)
        if plan.has_ghost:
            ops.halo_add(V_loc[:pe], V_loc[own:own + pe])
        return V_loc
    if fp32_payload:
        s32, r32 = scratch32 if scratch32 is not None else _buffers32(U_loc, pe, 2)
    # P^(t): first owned plane of U goes down, the ghost plane comes from above
    reqs = []
    if plan.down is not None:
        reqs.append(dist.isend(ops.pack_f32(s32, U_loc[:pe]) if fp32_payload else U_loc[:pe], plan.down))
    if plan.up is not None:
        reqs.append(dist.irecv(r32 if fp32_payload else U_loc[own:own + pe], plan.up))
    for r in reqs:
        r.wait()
    if fp32_payload and plan.up is not None:
        ops.unpack_f32(U_loc[own:own + pe], r32, False)
    if constraints is not None:                # C^(t)
        constraints.distribute(U_loc, nvec, homogeneous=True)
    ops.apply(U_loc, V_loc, nvec)
    if constraints is not None:                # C^(t)T
        constraints.distribute_transpose(V_loc, nvec)
    # P^(t)T: ghost plane of V goes up, the neighbour's comes from below and is added into the first plane
    if scratch is None and not fp32_payload:
        scratch = V_loc.new_empty(pe)
    reqs = []
    if plan.up is not None:
        reqs.append(dist.isend(ops.pack_f32(s32, V_loc[own:own + pe]) if fp32_payload else V_loc[own:own + pe], plan.up))
    if plan.down is not None:
        reqs.append(dist.irecv(r32 if fp32_payload else scratch[:pe], plan.down))
    for r in reqs:
        r.wait()
    if plan.down is not None:
        if fp32_payload:
            ops.unpack_f32(V_loc[:pe], r32, True)
        else:
            ops.halo_add(V_loc[:pe], scratch[:pe])
    return V_loc


TAG_U, TAG_V = 11, 12   # ghost values of U travel down, ghost rows of V travel up: two message kinds between a pair of tasks


def dd_apply_rank_batches(plan: SlabPlan, ops: LocalOps, U_list, V_list, nvec: int, dist, scratch_list=None,
                          fp32_payload: bool = False):
    """Algorithm 5: the multivector comes in n_b batches (one local multivector per batch, `nvec` columns
    each); while batch i_b is applied, the ghost exchange of batch i_b + 1 (Alg. 5 l.3-4, finished at l.8-9) and the halo
    add of batch i_b - 1 (l.5-6, finished at l.10-11) are in flight.  Messages between a pair of tasks are posted in
    the same order on both sides (U of the next batch first, then V of the previous one) and carry distinct tags.
    fp32_payload: the planes travel as FP32; the U and the V message of a step have their own send / receive buffers."""
    nb = len(U_list)
    pe = plan.plane_nodes * nvec
    own = plan.n_owned_planes * pe
    if plan.nslabs == 1:
        for U, V in zip(U_list, V_list):
            dd_apply_rank(plan, ops, U, V, nvec, dist)
        return V_list
    if fp32_payload:
        su32, ru32, sv32, rv32 = _buffers32(U_list[0], pe, 4)
    elif scratch_list is None:
        scratch_list = [V_list[0].new_empty(pe) for _ in range(2)]

    def start_u(i):       # P^(t) for batch i
        r = []
        if plan.down is not None:
            r.append(dist.isend(ops.pack_f32(su32, U_list[i][:pe]) if fp32_payload else U_list[i][:pe], plan.down, tag=TAG_U))
        if plan.up is not None:
            r.append(dist.irecv(ru32 if fp32_payload else U_list[i][own:own + pe], plan.up, tag=TAG_U))
        return r

    def finish_u(i, reqs):
        for r in reqs:
            r.wait()
        if fp32_payload and plan.up is not None:
            ops.unpack_f32(U_list[i][own:own + pe], ru32, False)

    def start_v(i):       # P^(t)T for batch i
        r = []
        if plan.up is not None:
            out = ops.pack_f32(sv32, V_list[i][own:own + pe]) if fp32_payload else V_list[i][own:own + pe]
            r.append(dist.isend(out, plan.up, tag=TAG_V))
        if plan.down is not None:
            r.append(dist.irecv(rv32 if fp32_payload else scratch_list[i & 1][:pe], plan.down, tag=TAG_V))
        return r

    def finish_v(i, reqs):
        for r in reqs:
            r.wait()
        if plan.down is not None:
            if fp32_payload:
                ops.unpack_f32(V_list[i][:pe], rv32, True)
            else:
                ops.halo_add(V_list[i][:pe], scratch_list[i & 1][:pe])

    finish_u(0, start_u(0))                               # Alg. 5 l.1
    for ib in range(nb):                                  # l.2
        ru = start_u(ib + 1) if ib + 1 < nb else []       # l.3-4
        rv = start_v(ib - 1) if ib > 0 else []            # l.5-6
        ops.apply(U_list[ib], V_list[ib], nvec)           # l.7
        if ib + 1 < nb:                                   # l.8-9
            finish_u(ib + 1, ru)
        if ib > 0:                                        # l.10-11
            finish_v(ib - 1, rv)
    finish_v(nb - 1, start_v(nb - 1))                     # l.12
    return V_list


def cheb_steps(m: int, a: float, b: float, a0: float):
    """The scalars of Alg. 6 l.2-16 (reading 10), in the paper's order and names: yields, for
    the first step, ("first", alpha1, alpha1 * alpha2) -- Y <- alpha1 A X + alpha1 alpha2 X -- and for every step
    d = 2..m ("step", alpha1, alpha2, -c alpha1) -- X <- alpha1 A Y + alpha2 X - c alpha1 Y, then swap."""
    if m < 1 or not (b > a) or not (a0 < a):
        raise ValueError("need m >= 1, b > a, a0 < a")
    e = (b - a) / 2.0
    c = (b + a) / 2.0
    sigma = e / (a0 - c)
    sigma1 = sigma
    gamma = 2.0 / sigma1
    alpha1 = sigma1 / e
    alpha2 = -c
    yield ("first", alpha1, alpha1 * alpha2)
    for _ in range(2, m + 1):
        sigma2 = 1.0 / (gamma - sigma)
        alpha1 = 2.0 * sigma2 / e
        alpha2 = -sigma * sigma2
        yield ("step", alpha1, alpha2, -(c * alpha1))
        sigma = sigma2


def dd_cheb_filter_rank(plan: SlabPlan, ops: LocalOps, X_loc, Y_loc, V_loc, nvec: int, m: int, a: float, b: float, a0: float,
                        dist, fp32_payload: bool = False):
    """One task of the Chebyshev filter on a decomposed mesh (the paper's multi-GPU eigenproblem runs):
    Alg. 6 l.2-17 with every product V = A U evaluated by dd_apply_rank (ghost exchange, fused local kernels, halo add)
    and the three-term update applied to the OWNED rows by fe_mf_axpby -- a slab context cannot fuse it into the kernel,
    because the ghost rows of V first travel to their owner.  X_loc / Y_loc / V_loc: local multivectors (owned planes +
    ghost plane; the ghost planes are scratch).  Returns (filtered block, iterate m - 1): the same two buffers, possibly
    exchanged (the paper's swap(X, Y), is an exchange of references here)."""
    own = plan.n_owned_planes * plan.plane_nodes * nvec
    X, Y = X_loc, Y_loc
    for step in cheb_steps(m, a, b, a0):
        if step[0] == "first":
            _, a1, a1a2 = step
            dd_apply_rank(plan, ops, X, V_loc, nvec, dist, fp32_payload=fp32_payload)
            ops.axpby(Y[:own], V_loc[:own], 0.0, a1)
            ops.axpby(Y[:own], X[:own], 1.0, a1a2)
        else:
            _, a1, a2, mca1 = step
            dd_apply_rank(plan, ops, Y, V_loc, nvec, dist, fp32_payload=fp32_payload)
            ops.axpby(X[:own], V_loc[:own], a2, a1)
            ops.axpby(X[:own], Y[:own], 1.0, mca1)
            X, Y = Y, X
    return Y, X


class SlabGroup:
    """All tasks of a decomposed mesh in ONE process on one device: the messages become device copies.  This is the
    form the path takes on a single GPU (tests, bench); with one process per GPU use dd_apply_rank."""

    def __init__(self, w, nslabs: int, device: int = 0, make_ops: Optional[Callable] = None):
        from . import inputs
        periodic = w.bc == inputs.BC_PERIODIC
        self.w, self.nslabs = w, nslabs
        self.plans = [make_plan(w.ncells, w.p, periodic, nslabs, t) for t in range(nslabs)]
        self.ops, self.ctxs = [], []
        for pl in self.plans:
            if make_ops is None:
                o, ctx = device_ops(w, pl, device)
                self.ctxs.append(ctx)
            else:
                o = make_ops(w, pl)
            self.ops.append(o)

    def scatter(self, X, nvec: int):
        """Global multivector (flat, nd_z planes) -> list of local multivectors (owned planes + ghost plane left unset)."""
        out = []
        for pl in self.plans:
            pe = pl.plane_nodes * nvec
            U = X.new_empty(pl.nplanes * pe)
            first = pl.z0 * pl.p
            U[:pl.n_owned_planes * pe].copy_(X[first * pe:(first + pl.n_owned_planes) * pe])
            out.append(U)
        return out

    def gather(self, V_locs, nvec: int, out):
        """Owned planes of every task -> global multivector."""
        for pl, V in zip(self.plans, V_locs):
            pe = pl.plane_nodes * nvec
            first = pl.z0 * pl.p
            out[first * pe:(first + pl.n_owned_planes) * pe].copy_(V[:pl.n_owned_planes * pe])
        return out

    def apply(self, U_locs, V_locs, nvec: int, fp32_payload: bool = False, constraints=None):
        """V^(t) for every task, ghost planes exchanged and added: on return the owned planes of V_locs hold A U.
        fp32_payload: every plane that crosses a task boundary goes through an FP32 message buffer (pack / unpack).
        constraints: one C^(t) per task (see dd_apply_rank): the owned planes then hold C^T A C U."""
        plans = self.plans
        fp32 = fp32_payload and self.nslabs > 1
        if fp32:
            (m32,) = _buffers32(U_locs[0], plans[0].plane_nodes * nvec, 1)
        for pl, U in zip(plans, U_locs):                      # P^(t)
            if pl.has_ghost:
                pe = pl.plane_nodes * nvec
                own = pl.n_owned_planes * pe
                if fp32:
                    self.ops[pl.up].pack_f32(m32, U_locs[pl.up][:pe])
                    self.ops[pl.rank].unpack_f32(U[own:own + pe], m32, False)
                else:
                    U[own:own + pe].copy_(U_locs[pl.up][:pe])
        for t, (o, U, V) in enumerate(zip(self.ops, U_locs, V_locs)):     # C^(t)T A^(t) C^(t)
            if constraints is not None:
                constraints[t].distribute(U, nvec, homogeneous=True)
            o.apply(U, V, nvec)
            if constraints is not None:
                constraints[t].distribute_transpose(V, nvec)
        # P^(t)T: every first plane is final after the local applies only in its OWN task's sum, so the adds are
        # independent of one another (a task's ghost plane is never another add's destination)
        for pl, V in zip(plans, V_locs):
            if pl.has_ghost:
                pe = pl.plane_nodes * nvec
                own = pl.n_owned_planes * pe
                if fp32:
                    self.ops[pl.rank].pack_f32(m32, V[own:own + pe])
                    self.ops[pl.up].unpack_f32(V_locs[pl.up][:pe], m32, True)
                else:
                    self.ops[pl.up].halo_add(V_locs[pl.up][:pe], V[own:own + pe])
        return V_locs

    def cheb_filter(self, X_locs, Y_locs, V_locs, nvec: int, m: int, a: float, b: float, a0: float, fp32_payload: bool = False):
        """dd_cheb_filter_rank for all tasks of the group.  Returns (filtered blocks, iterates m - 1): the two lists of
        buffers, possibly exchanged."""
        owns = [pl.n_owned_planes * pl.plane_nodes * nvec for pl in self.plans]
        X, Y = X_locs, Y_locs
        for step in cheb_steps(m, a, b, a0):
            if step[0] == "first":
                _, a1, a1a2 = step
                self.apply(X, V_locs, nvec, fp32_payload=fp32_payload)
                for o, own, x, y, v in zip(self.ops, owns, X, Y, V_locs):
                    o.axpby(y[:own], v[:own], 0.0, a1)
                    o.axpby(y[:own], x[:own], 1.0, a1a2)
            else:
                _, a1, a2, mca1 = step
                self.apply(Y, V_locs, nvec, fp32_payload=fp32_payload)
                for o, own, x, y, v in zip(self.ops, owns, X, Y, V_locs):
                    o.axpby(x[:own], v[:own], a2, a1)
                    o.axpby(x[:own], y[:own], 1.0, mca1)
                X, Y = Y, X
        return Y, X
