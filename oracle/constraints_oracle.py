"""CPU oracle of the constraint matrices C^(t), C^(t)T (section 3.2.2) -- TEST
INFRASTRUCTURE, NOT THE PRODUCT (same rules as fe_oracle.py: only tests/, smoke() and bench.py's cpu_baseline legs may
import it).

The paper stores the constraints "as multiple sets, and each set I comprises four arrays": the master node indices,
the slave node indices, the weight matrix W_I and the inhomogeneities b_I of the slaves.  The action of C
on a multivector is, set by set,

    U_{S_I}  <-  W_I U_{M_I} + b_I            (extract the master rows, one dense product, add b_I, copy to the slave rows)

and "the action of C^T is evaluated in the similar manner": C is the matrix with C[s, m] = W_I[s, m] for the
slaves, a zero column for every slave and the identity elsewhere, so

    V_{M_I}  <-  V_{M_I} + W_I^T V_{S_I},     V_{S_I}  <-  0.

Dirichlet conditions are sets with no masters ("the master index matrix and weight matrix are empty").

Reading (the paper is silent; reading 19): the sets are CLOSED -- no slave of any set is a master of any set,
and every slave belongs to exactly one set (deal.II resolves chains when the constraints are closed).  The order of
the sets is then immaterial and C is idempotent.  `check_closed` enforces it.

Everything is written out as the definition: row gathers, one matrix product per set, row scatters.  Pins
(tests/test_oracle_constraints.py): <C U, V> = <U, C^T V> (adjointness, homogeneous part); C C U = C U; C against the
explicit sparse matrix built entry by entry; hanging-node weights reproduce every polynomial of degree <= p on the
coarse face and have unit row sums; a periodic mesh IS an open slab with the constraint "top plane = bottom plane"
(C^T A_open C = the periodic operator of fe_oracle, through dd_oracle.slab_apply) and a Dirichlet mesh IS the same
slab with master-less sets on the two end planes.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass
class ConstraintSet:
    """One set I of PAPER.md:290: masters [nm], slaves [ns], W [ns][nm], b [ns]."""
    masters: np.ndarray
    slaves: np.ndarray
    W: np.ndarray
    b: np.ndarray

    def __post_init__(self):
        self.masters = np.asarray(self.masters, dtype=np.int64).reshape(-1)
        self.slaves = np.asarray(self.slaves, dtype=np.int64).reshape(-1)
        self.W = np.asarray(self.W, dtype=np.float64).reshape(len(self.slaves), len(self.masters))
        self.b = np.zeros(len(self.slaves)) if self.b is None else np.asarray(self.b, dtype=np.float64).reshape(-1)
        if len(self.b) != len(self.slaves):
            raise ValueError("one inhomogeneity per slave")


def check_closed(sets, ndof: int) -> None:
    """Every index in range; every slave in exactly one set; no slave is a master (reading 19)."""
    seen = np.zeros(ndof, dtype=np.int64)
    for I in sets:
        for idx in (I.masters, I.slaves):
            if len(idx) and (idx.min() < 0 or idx.max() >= ndof):
                raise ValueError("node index out of range")
        np.add.at(seen, I.slaves, 1)
    if seen.max(initial=0) > 1:
        raise ValueError("a slave belongs to two sets (or twice to one)")
    for I in sets:
        if len(I.masters) and seen[I.masters].any():
            raise ValueError("a slave is a master: the constraints are not closed")


def distribute(sets, U: np.ndarray, homogeneous: bool = False) -> np.ndarray:
    """C U (+ the inhomogeneities): U_{S_I} = W_I U_{M_I} + b_I for every set."""
    U = np.array(U, dtype=np.float64, copy=True)
    check_closed(sets, U.shape[0])
    for I in sets:
        US = I.W @ U[I.masters] if len(I.masters) else np.zeros((len(I.slaves), U.shape[1]))
        if not homogeneous:
            US = US + I.b[:, None]
        U[I.slaves] = US
    return U


def distribute_transpose(sets, V: np.ndarray) -> np.ndarray:
    """C^T V: V_{M_I} += W_I^T V_{S_I}, then V_{S_I} = 0."""
    V = np.array(V, dtype=np.float64, copy=True)
    check_closed(sets, V.shape[0])
    for I in sets:
        if len(I.masters):
            np.add.at(V, I.masters, I.W.T @ V[I.slaves])       # a master may occur in several sets: accumulate
        V[I.slaves] = 0.0
    return V


def hanging_face_weights(p: int, child: tuple[int, int]) -> np.ndarray:
    """W of a hanging FACE (the locally dense constraints of PAPER.md:290, "interpolation along faces"): a coarse face
    with (p+1)^2 master nodes at the GLL tensor grid of [-1,1]^2 borders a refined cell whose child face `child`
    = (c1, c2) in {0,1}^2 covers the quadrant [c1-1, c1] x [c2-1, c2]; the child's (p+1)^2 nodes take the values of the
    coarse face's polynomial:  W[(j2, j1), (i2, i1)] = l_i1(x_j1) l_i2(y_j2),  x_j = (xi_j + 2 c1 - 1) / 2."""
    from .fe_oracle import gll_nodes, lagrange_values
    xi = gll_nodes(p)
    L1 = lagrange_values(xi, (xi + 2 * child[0] - 1) / 2)      # [j][i] = l_i(x_j)
    L2 = lagrange_values(xi, (xi + 2 * child[1] - 1) / 2)
    n = p + 1
    W = np.einsum("bi,aj->abji", L1, L2)                        # [j2][j1][i2][i1] = L2[j2][i2] L1[j1][i1]
    return np.asarray(W, dtype=np.float64).reshape(n * n, n * n)
