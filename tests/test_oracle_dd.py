"""Pins of the domain-decomposed oracle (oracle/dd_oracle.py; Alg. 5): the
partitioner's bookkeeping, and the exact identity sum_t P^(t)T A^(t) P^(t) U = A U against the single-domain oracle."""
import numpy as np
import pytest

from oracle import dd_oracle as ddo
from oracle import fe_oracle as orc
from paper_2208_07129_b200 import inputs


def test_slab_layers_cover_the_mesh():
    for ncz in (3, 8, 13):
        for ns in range(1, ncz + 1):
            lay = ddo.slab_layers(ncz, ns)
            assert lay[0][0] == 0 and lay[-1][1] == ncz
            assert all(a[1] == b[0] for a, b in zip(lay, lay[1:]))
            sizes = [z1 - z0 for z0, z1 in lay]
            assert max(sizes) - min(sizes) <= 1 and min(sizes) >= 1
    with pytest.raises(ValueError):
        ddo.slab_layers(3, 4)


@pytest.mark.parametrize("bc", ["periodic", "dirichlet"])
@pytest.mark.parametrize("nslabs", [1, 2, 3, 5])
def test_every_node_has_one_owner_and_ghosts_are_one_plane(bc, nslabs):
    """m_loc^(t) partition the DoFs; m_ghost^(t) = one node plane ('locally-owned ... followed by ghost')."""
    mesh = orc.Mesh((2, 3, 5), 3, bc)
    owners = np.zeros(mesh.ndof, dtype=int)
    plane = mesh.nd[0] * mesh.nd[1]
    for t, (z0, z1) in enumerate(ddo.slab_layers(5, nslabs)):
        rows, n_owned = ddo.slab_rows(mesh, z0, z1)
        owners[rows[:n_owned]] += 1
        nghost = len(rows) - n_owned
        last_dirichlet = bc == "dirichlet" and z1 == 5
        assert nghost == (0 if last_dirichlet else plane)
        assert len(rows) == ((z1 - z0) * 3 + 1) * plane
        if nghost:   # the ghost plane is the first owned plane of the next task (cyclically)
            nz0 = ddo.slab_layers(5, nslabs)[(t + 1) % nslabs][0]
            nrows, _ = ddo.slab_rows(mesh, nz0, ddo.slab_layers(5, nslabs)[(t + 1) % nslabs][1])
            assert np.array_equal(rows[n_owned:], nrows[:plane])
    assert np.all(owners == 1)


@pytest.mark.parametrize("bc", ["periodic", "dirichlet"])
@pytest.mark.parametrize("p,nc", [(2, (2, 3, 5)), (4, (2, 2, 4)), (6, (2, 2, 3))])
def test_decomposed_apply_is_the_single_domain_apply(bc, p, nc):
    """Exact identity (up to summation order, 1e-14) for every admissible number of slabs; and each communication step
    is needed: without the ghost exchange or without the halo add the result is wrong at the cut planes."""
    mesh = orc.Mesh(nc, p, bc, (0.0, -1.0, 2.0), (1.0, 0.5, 4.4))
    op = orc.Operator(mesh, 0.7)
    rng = np.random.default_rng(11 + p)
    X = rng.uniform(-1, 1, (mesh.ndof, 3))
    Y = op.apply(X)
    scale = np.abs(Y).max()
    for ns in range(1, nc[2] + 1):
        assert np.abs(ddo.dd_apply(op, X, ns) - Y).max() <= 1e-14 * scale
    ns = 2
    assert np.abs(ddo.dd_apply(op, X, ns, exchange_ghosts=False) - Y).max() > 1e-3 * scale
    assert np.abs(ddo.dd_apply(op, X, ns, halo_add=False) - Y).max() > 1e-3 * scale


def test_decomposed_apply_on_the_perturbed_mesh():
    """Per-q-point geometry (config 3's recipe at a small size): the cells of a slab keep their own metric."""
    w = inputs.configs()[3].scaled(3, nvec=2)
    mesh = orc.Mesh(w.ncells, 3, "periodic", w.box_lo, w.box_hi,
                    vertices=inputs.perturbed_vertices(w.ncells, w.box_lo, w.box_hi, 0.15, 99))
    op = orc.Operator(mesh, 1.0)
    X = inputs.multivector(5, mesh.ndof, 2)
    Y = op.apply(X)
    for ns in (2, 3):
        assert np.abs(ddo.dd_apply(op, X, ns) - Y).max() <= 1e-14 * np.abs(Y).max()
