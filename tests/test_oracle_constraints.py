"""Pins of the constraint oracle (oracle/constraints_oracle.py; section 3.2.2): what the mathematics
fixes about C and C^T, the hanging-node weights, and the two constraints the FE oracle already contains in another
form -- periodicity and the Dirichlet condition."""
import numpy as np
import pytest

from oracle import constraints_oracle as co
from oracle import dd_oracle as ddo
from oracle import fe_oracle as orc


def random_sets(rng, ndof, nsets, inhomogeneous=True):
    """Closed sets on a random node subset: slaves disjoint from everything, masters may be shared between sets and
    one set has no masters (a Dirichlet set)."""
    perm = rng.permutation(ndof)
    nslave_total = ndof // 3
    slaves_pool, masters_pool = perm[:nslave_total], perm[nslave_total:]
    cuts = np.sort(rng.choice(np.arange(1, nslave_total), nsets - 1, replace=False))
    sets = []
    for k, sl in enumerate(np.split(slaves_pool, cuts)):
        nm = 0 if k == 0 else int(rng.integers(1, 9))
        ms = rng.choice(masters_pool, nm, replace=False)
        W = rng.uniform(-1, 1, (len(sl), nm))
        b = rng.uniform(-1, 1, len(sl)) if inhomogeneous else None
        sets.append(co.ConstraintSet(ms, sl, W, b))
    return sets


def explicit_matrix(sets, ndof):
    C = np.eye(ndof)
    for I in sets:
        C[I.slaves, :] = 0.0
    for I in sets:
        for a, s in enumerate(I.slaves):
            for c, m in enumerate(I.masters):
                C[s, m] += I.W[a, c]
    return C


def test_c_and_ct_against_the_explicit_matrix_adjointness_idempotence():
    rng = np.random.default_rng(3)
    ndof, nvec = 120, 3
    sets = random_sets(rng, ndof, 6)
    C = explicit_matrix(sets, ndof)
    U = rng.uniform(-1, 1, (ndof, nvec)); V = rng.uniform(-1, 1, (ndof, nvec))
    CU = co.distribute(sets, U, homogeneous=True)
    CtV = co.distribute_transpose(sets, V)
    assert np.abs(CU - C @ U).max() <= 1e-14
    assert np.abs(CtV - C.T @ V).max() <= 1e-14
    assert abs(np.sum(CU * V) - np.sum(U * CtV)) <= 1e-12                                   # <C U, V> = <U, C^T V>
    bvec = np.zeros(ndof)
    for I in sets:
        bvec[I.slaves] = I.b
    CUb = co.distribute(sets, U)
    assert np.abs(CUb - (C @ U + bvec[:, None])).max() <= 1e-14                            # the inhomogeneities
    assert np.array_equal(co.distribute(sets, CUb), CUb)                                    # C is idempotent (closed sets)
    for I in sets:
        assert np.all(CtV[I.slaves] == 0.0)                                                 # zero columns of C


def test_unclosed_sets_are_refused():
    with pytest.raises(ValueError):     # a slave that is a master
        co.distribute([co.ConstraintSet([1], [2], [[1.0]], None), co.ConstraintSet([2], [3], [[1.0]], None)], np.zeros((5, 1)))
    with pytest.raises(ValueError):     # a slave in two sets
        co.distribute([co.ConstraintSet([1], [2], [[1.0]], None), co.ConstraintSet([0], [2], [[1.0]], None)], np.zeros((5, 1)))
    with pytest.raises(ValueError):     # out of range
        co.distribute([co.ConstraintSet([7], [2], [[1.0]], None)], np.zeros((5, 1)))


@pytest.mark.parametrize("p", [1, 2, 3, 6, 8])
def test_hanging_face_weights_reproduce_the_coarse_polynomial(p):
    """The slave values are the coarse face's polynomial at the child nodes: exact for every tensor polynomial of
    degree <= p; rows sum to one; a child node that coincides with a coarse node copies it."""
    xi = np.asarray(orc.gll_nodes(p), dtype=np.float64)
    rng = np.random.default_rng(p)
    coef = rng.uniform(-1, 1, (p + 1, p + 1))
    poly = lambda x, y: np.polynomial.polynomial.polyval2d(x, y, coef)     # noqa: E731
    X, Y = np.meshgrid(xi, xi, indexing="xy")                              # [i2][i1]: x varies fastest
    coarse = poly(X, Y).reshape(-1)
    for child in [(0, 0), (1, 0), (0, 1), (1, 1)]:
        W = co.hanging_face_weights(p, child)
        xc, yc = (xi + 2 * child[0] - 1) / 2, (xi + 2 * child[1] - 1) / 2
        Xc, Yc = np.meshgrid(xc, yc, indexing="xy")
        assert np.abs(W @ coarse - poly(Xc, Yc).reshape(-1)).max() <= 1e-13
        assert np.abs(W.sum(axis=1) - 1).max() <= 1e-14
        n = p + 1
        corner = (child[1] * p) * n + child[0] * p          # the child's outer corner IS the coarse face's corner
        e = np.zeros(n * n); e[corner] = 1.0
        assert np.abs(W[corner] - e).max() <= 1e-15


@pytest.mark.parametrize("p,nc", [(2, (2, 3, 3)), (4, (2, 2, 2))])
def test_periodicity_is_a_constraint_on_an_open_slab(p, nc):
    """C^T A_open C = the periodic operator: the whole periodic mesh as ONE slab (its top plane is a copy of plane 0),
    the copy expressed as a constraint set with W = identity."""
    mesh = orc.Mesh(nc, p, "periodic", (0, 0, 0), (1.0, 1.2, 0.9))
    op = orc.Operator(mesh, 0.6)
    rng = np.random.default_rng(p)
    X = rng.uniform(-1, 1, (mesh.ndof, 2))
    plane = mesh.nd[0] * mesh.nd[1]
    nloc = mesh.ndof + plane
    top = np.arange(mesh.ndof, nloc)
    sets = [co.ConstraintSet(np.arange(plane), top, np.eye(plane), None)]
    U = np.vstack([X, rng.uniform(-9, 9, (plane, 2))])                     # the slave rows hold garbage before C
    V = co.distribute_transpose(sets, ddo.slab_apply(op, 0, nc[2], co.distribute(sets, U)))
    Y = op.apply(X)
    assert np.abs(V[:mesh.ndof] - Y).max() <= 1e-13 * np.abs(Y).max()
    assert np.all(V[top] == 0.0)


def test_dirichlet_is_a_masterless_constraint_on_an_open_slab():
    """Dirichlet conditions through the same framework, with empty master arrays.  The middle layers of a
    taller Dirichlet mesh form a slab whose end planes are cut planes (open); with master-less sets on those two planes
    the slab operator is the Dirichlet operator of the shorter mesh."""
    p, ncx, ncy, ncz, h = 3, 2, 2, 4, 0.5
    tall = orc.Mesh((ncx, ncy, ncz), p, "dirichlet", (0, 0, 0), (1.0, 1.0, ncz * h))
    short = orc.Mesh((ncx, ncy, ncz - 2), p, "dirichlet", (0, 0, h), (1.0, 1.0, (ncz - 1) * h))
    op_tall, op_short = orc.Operator(tall, 0.9), orc.Operator(short, 0.9)
    plane = short.nd[0] * short.nd[1]
    rng = np.random.default_rng(8)
    X = rng.uniform(-1, 1, (short.ndof, 2))
    ends = np.concatenate([np.arange(plane), np.arange(short.ndof - plane, short.ndof)])
    sets = [co.ConstraintSet([], ends, np.zeros((len(ends), 0)), None)]
    V = co.distribute_transpose(sets, ddo.slab_apply(op_tall, 1, ncz - 1, co.distribute(sets, X)))
    Y = op_short.apply(X)
    assert np.abs(V - Y).max() <= 1e-13 * np.abs(Y).max()
    # and without the sets the open slab is NOT the Dirichlet operator
    assert np.abs(ddo.slab_apply(op_tall, 1, ncz - 1, X) - Y).max() > 1e-3 * np.abs(Y).max()
