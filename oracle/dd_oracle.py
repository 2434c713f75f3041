"""CPU oracle of the domain-decomposed apply -- TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules
as fe_oracle.py: only tests/, smoke() and bench.py's cpu_baseline legs may import it).

The paper distributes the mesh over tasks t; a task holds its locally-owned DoFs followed by the "ghost" DoFs on the
shared subdomain boundary that another task owns, and evaluates (Eq. 6 / 16)

    V = sum_t  P^(t)T [ C^(t)T ( sum_{e in E_t} Q^(e,t)T A^(e) Q^(e,t) ) C^(t) ] P^(t) U

P^(t) = the partitioner: extraction of task t's owned + ghost rows (the ghost rows arrive by point-to-point messages,
PAPER.md:746, Alg. 5 l.1/3/8); P^(t)T = the reverse: ghost rows of V^(t) are sent to their owner and ADDED (Alg. 5
l.5/10/12).  Here the subdomains are z-SLABS of the structured mesh (the simplest instance: every task has at most
two neighbours, or itself across the periodic boundary):

    task t owns the cell layers z0_t <= ez < z1_t and the node planes  z0_t p <= iz < z1_t p  (the last task of a
    Dirichlet mesh also owns the boundary plane ncz p); its one ghost plane is  iz = z1_t p  (owned by task t+1; on a
    periodic mesh the last task's ghost plane is plane 0 of task 0).  Local row order = plane order: owned planes
    first, then the ghost plane -- the layout of PAPER.md:748 ("m_loc followed by m_ghost").

Everything is written out with index arrays (P^(t) as a row list), cell by cell, through fe_oracle's element
matrices: no kernels, no fusion.  Pins (tests/test_oracle_dd.py): every global node has exactly one owner; the ghost
count is one node plane; sum_t P^(t)T V^(t) reproduces fe_oracle.Operator.apply for any number of slabs on periodic,
Dirichlet and perturbed meshes (an exact identity up to summation order); with the ghost exchange or the halo add
left out the identity fails at the cut planes.

Mixed-precision boundary payload ("the boundary data communicated is recast as FP32 floats"): with
`fp32_payload` every value that crosses a task boundary -- the ghost rows of U on their way in, the ghost rows of V^(t)
on their way back -- is rounded to IEEE binary32 (round to nearest even) and widened again; everything a task computes
stays FP64.  A single task exchanges nothing, so nothing is rounded.  Pins: the deviation from the exact apply lives
only in the cell layer under a cut plane, on the cut plane itself it is the rounding error of the exact ghost row when
U is FP32-representable, and it is of the size of the FP32 unit roundoff.

dd_constrained_apply: Eq. 17 in full, with the constraint matrices C^(t), C^(t)T of oracle/constraints_oracle.py around the
local cell loop.  Pin: equal to C^T A C of the undecomposed mesh (constraints_oracle on the global rows around
fe_oracle.Operator.apply) when every set lies inside one task's local rows; a set that straddles a cut is refused.

dd_chebyshev_filter: the filter recurrence of fe_oracle.chebyshev_filter with the decomposed apply as its operator.  Pins:
equal to the single-domain filter for every slab count (1e-12: m steps of summation-order differences, amplified by the
filter's growth outside [a, b]); with the FP32 payload the deviation stays at the FP32 level times that growth.
"""
from __future__ import annotations

import numpy as np


def slab_layers(ncz: int, nslabs: int):
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


def slab_rows(mesh, z0: int, z1: int):
    """Global rows of task t's local multivector, in local order: node planes z0 p .. z1 p (inclusive), wrapped on a
    periodic mesh.  Returns (rows, n_owned): the first n_owned rows are locally owned, the rest is the ghost plane."""
    p, (ndx, ndy, ndz) = mesh.p, mesh.nd
    plane = ndx * ndy
    planes = [iz % ndz if mesh.bc == "periodic" else iz for iz in range(z0 * p, z1 * p + 1)]
    rows = np.concatenate([iz * plane + np.arange(plane) for iz in planes])
    last_is_owned = mesh.bc != "periodic" and z1 == mesh.ncells[2]      # the physical boundary plane
    n_owned = len(rows) if last_is_owned else len(rows) - plane
    return rows, n_owned


def slab_apply(op, z0: int, z1: int, U_loc: np.ndarray) -> np.ndarray:
    """V^(t) = C^(t)T ( sum_{e in E_t} Q^T A^(e) Q ) C^(t) U^(t) on the cells of layers z0 <= ez < z1, in the LOCAL
    row order of slab_rows.  Constraints are those of the global mesh restricted to the task (Dirichlet boundary
    nodes of the physical boundary only: a cut plane is not a boundary)."""
    m = op.mesh
    p, (ndx, ndy, ndz) = m.p, m.nd
    plane = ndx * ndy
    V = np.zeros_like(U_loc)
    for ez in range(z0, z1):
        for ey in range(m.ncells[1]):
            for ex in range(m.ncells[0]):
                idx, mask = m.cell_dofs(ex, ey, ez)              # global rows (wrapped on periodic meshes)
                giz = idx // plane
                # local plane = global plane - z0 p; the wrapped top plane of a periodic mesh is the ghost plane
                liz = giz - z0 * p
                if m.bc == "periodic":
                    liz = np.where(liz < 0, liz + ndz, liz)
                    if ez == z1 - 1:                              # top layer: its top nodes live in the ghost plane
                        top = (ez * p + m._i[2]) == z1 * p
                        liz = np.where(top, (z1 - z0) * p, liz)
                lidx = liz * plane + idx % plane
                U = U_loc[lidx]
                if mask is not None:
                    U[mask] = 0.0
                W = op.cell_apply(ex, ey, ez, U)
                if mask is not None:
                    W[mask] = 0.0
                V[lidx] += W
    return V


def round_fp32(a: np.ndarray) -> np.ndarray:
    """The FP32 payload of PAPER.md:752: FP64 -> binary32 (round to nearest even) -> FP64."""
    return np.asarray(a, dtype=np.float64).astype(np.float32).astype(np.float64)


def dd_apply(op, X: np.ndarray, nslabs: int, exchange_ghosts: bool = True, halo_add: bool = True,
             fp32_payload: bool = False) -> np.ndarray:
    """V = sum_t P^(t)T V^(t), V^(t) = A^(t) P^(t) U.  exchange_ghosts / halo_add exist for the pins only (what breaks
    without each communication step); fp32_payload: the communicated rows travel as FP32."""
    m = op.mesh
    X = np.asarray(X, dtype=np.float64)
    V = np.zeros_like(X)
    for (z0, z1) in slab_layers(m.ncells[2], nslabs):
        rows, n_owned = slab_rows(m, z0, z1)
        U_loc = X[rows].copy()                                   # P^(t) U: owned rows + received ghost rows
        if not exchange_ghosts:
            U_loc[n_owned:] = 0.0
        elif fp32_payload and nslabs > 1:
            U_loc[n_owned:] = round_fp32(U_loc[n_owned:])        # the ghost rows arrived as FP32
        V_loc = slab_apply(op, z0, z1, U_loc)
        if fp32_payload and nslabs > 1:
            V_loc[n_owned:] = round_fp32(V_loc[n_owned:])        # the ghost rows leave as FP32
        if halo_add:
            np.add.at(V, rows, V_loc)                            # P^(t)T: owned rows stay, ghost rows go to their owner
        else:
            np.add.at(V, rows[:n_owned], V_loc[:n_owned])
    return V


def dd_chebyshev_filter(op, X: np.ndarray, nslabs: int, m: int, a: float, b: float, a0: float,
                        fp32_payload: bool = False) -> np.ndarray:
    """The Chebyshev filter (Alg. 6 l.2-17) with EVERY operator application evaluated in decomposed
    form, V = sum_t P^(t)T A^(t) P^(t) U (the paper's multi-GPU eigenproblem runs): the recurrence is
    fe_oracle.chebyshev_filter's, line by line; only the operator is replaced.  Without the FP32 payload this equals the
    single-domain filter up to summation order (pinned in tests/test_oracle_dd.py); with it every step's boundary planes are
    rounded to binary32 on their way across a cut."""
    from .fe_oracle import chebyshev_filter
    return chebyshev_filter(lambda V: dd_apply(op, V, nslabs, fp32_payload=fp32_payload), X, m, a, b, a0)


# ---- Eq. 17 in full: the constraint matrices inside the decomposed apply ----------------------------------------------

def restrict_sets(sets, rows: np.ndarray):
    """C^(t): the global constraint sets (oracle/constraints_oracle.ConstraintSet, global row indices) restricted to the
    local rows of a task.  A set takes part in task t if one of its slaves is a local row; then ALL its slaves and
    masters must be local rows (the locally dense sets of PAPER.md:290 live on one face / edge; a set that straddles a cut
    would need masters the task does not hold) -- otherwise ValueError.  A global row on a cut plane is local to two tasks:
    both get the set."""
    from .constraints_oracle import ConstraintSet
    pos = {}
    for k, r in enumerate(rows):                      # a single periodic task holds plane 0 twice (first plane and ghost plane)
        pos.setdefault(int(r), []).append(k)
    out = []
    for I in sets:
        here = [int(s) in pos for s in I.slaves]
        if not any(here):
            continue
        nodes = [int(v) for v in np.concatenate([I.masters, I.slaves])]
        if not all(v in pos for v in nodes):
            raise ValueError("a constraint set straddles a subdomain boundary")
        copies = {len(pos[v]) for v in nodes}
        if len(copies) != 1:
            raise ValueError("a constraint set mixes rows the task holds once and rows it holds twice")
        for c in range(copies.pop()):                 # one local set per copy
            out.append(ConstraintSet([pos[int(m_)][c] for m_ in I.masters], [pos[int(s)][c] for s in I.slaves], I.W, I.b))
    return out


def dd_constrained_apply(op, X: np.ndarray, nslabs: int, sets) -> np.ndarray:
    """Eq. 17:  V = sum_t P^(t)T C^(t)T ( sum_{e in E_t} Q^T A^(e) Q ) C^(t) P^(t) U, the homogeneous part
    of the constraints (an operator apply).  Step by step per task: extract owned + ghost rows, distribute, the local cell
    loop, distribute-transpose, add into the global rows."""
    from .constraints_oracle import distribute, distribute_transpose
    m = op.mesh
    X = np.asarray(X, dtype=np.float64)
    V = np.zeros_like(X)
    for (z0, z1) in slab_layers(m.ncells[2], nslabs):
        rows, _ = slab_rows(m, z0, z1)
        loc = restrict_sets(sets, rows)
        U_loc = distribute(loc, X[rows], homogeneous=True)
        V_loc = distribute_transpose(loc, slab_apply(op, z0, z1, U_loc))
        np.add.at(V, rows, V_loc)
    return V
