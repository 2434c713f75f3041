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


@pytest.mark.parametrize("bc", ["periodic", "dirichlet"])
def test_fp32_payload_deviates_only_under_the_cut_planes(bc):
    """PAPER.md:752 (FP32 boundary payload).  What the mathematics fixes: (i) a single task exchanges nothing: no
    deviation; (ii) the deviation from the exact apply is confined to the cell layer under each cut plane (rounded ghost
    values of U enter only the cells that touch the ghost plane; rounded ghost rows of V land on the cut plane);
    (iii) it has the size of the FP32 unit roundoff 2^-24, not of FP64 and not O(1); (iv) when U is itself
    FP32-representable the inbound rounding is the identity: the deviation then sits on the cut planes only and there it
    is exactly fl32(g) - g for the ghost row g of the exact local product, computed here from slab_apply directly."""
    p, nc, ns = 3, (2, 2, 5), 2
    mesh = orc.Mesh(nc, p, bc)
    op = orc.Operator(mesh, 0.7)
    rng = np.random.default_rng(5)
    X = rng.uniform(-1, 1, (mesh.ndof, 2))
    Y = ddo.dd_apply(op, X, ns)
    scale = np.abs(Y).max()
    assert np.array_equal(ddo.dd_apply(op, X, 1, fp32_payload=True), ddo.dd_apply(op, X, 1))          # (i)
    D = ddo.dd_apply(op, X, ns, fp32_payload=True) - Y
    plane = mesh.nd[0] * mesh.nd[1]
    ndz = mesh.nd[2]
    layers = ddo.slab_layers(nc[2], ns)
    allowed = np.zeros(ndz, dtype=bool)
    cuts = []
    for (z0, z1) in layers:
        if bc == "dirichlet" and z1 == nc[2]:
            continue                                                   # the physical boundary is not a cut
        cuts.append((z0, z1))
        for iz in range((z1 - 1) * p, z1 * p + 1):
            allowed[iz % ndz] = True
    dev = np.abs(D).reshape(ndz, plane * 2).max(axis=1)
    assert np.all(dev[~allowed] == 0.0)                                                                # (ii)
    assert dev[allowed].min() > 0.0
    assert 1e-10 * scale < dev.max() < 100 * 2.0 ** -24 * scale                                        # (iii)
    # (iv)
    X32 = ddo.round_fp32(X)
    Y32 = ddo.dd_apply(op, X32, ns)
    D32 = ddo.dd_apply(op, X32, ns, fp32_payload=True) - Y32
    on_cut = np.zeros(ndz, dtype=bool)
    expect = np.zeros_like(Y32)
    for (z0, z1) in cuts:
        on_cut[(z1 * p) % ndz] = True
        rows, n_owned = ddo.slab_rows(mesh, z0, z1)
        g = ddo.slab_apply(op, z0, z1, X32[rows].copy())[n_owned:]
        expect[rows[n_owned:]] += ddo.round_fp32(g) - g
    dev32 = np.abs(D32).reshape(ndz, plane * 2).max(axis=1)
    assert np.all(dev32[~on_cut] == 0.0) and np.all(dev32[on_cut] > 0.0)
    assert np.abs(D32 - expect).max() <= 4e-16 * scale
    if bc == "dirichlet":                                              # boundary rows stay exactly zero
        ix, iy, iz = np.meshgrid(*[np.arange(n) for n in mesh.nd], indexing="ij")
        bnd = (ix == 0) | (ix == mesh.nd[0] - 1) | (iy == 0) | (iy == mesh.nd[1] - 1) | (iz == 0) | (iz == ndz - 1)
        rows = (ix + mesh.nd[0] * (iy + mesh.nd[1] * iz))[bnd]
        assert np.all(ddo.dd_apply(op, X, ns, fp32_payload=True)[rows] == 0.0)


@pytest.mark.parametrize("bc", ["periodic", "dirichlet"])
def test_decomposed_chebyshev_filter_is_the_single_domain_filter(bc):
    """Alg. 6 with the decomposed operator: the same polynomial of the same matrix, whatever the number of tasks.  The
    spectrum bound comes from the oracle's Lanczos; [a, b] covers the upper 60 % of the spectrum (damped), the scaled
    filter is 1 at a0."""
    p, nc, m = 3, (2, 2, 4), 7
    mesh = orc.Mesh(nc, p, bc, (0.0, 0.0, 0.0), (1.0, 1.2, 2.0))
    op = orc.Operator(mesh, 0.7)
    X = inputs.multivector(91, mesh.ndof, 3)
    b = orc.lanczos_upper_bound(op.apply, inputs.uniform_pm1(92, 0, mesh.ndof), 10)
    a, a0 = 0.4 * b, 0.0
    Y = orc.chebyshev_filter(op.apply, X, m, a, b, a0)
    assert np.abs(Y - X).max() > 0.1 * np.abs(X).max()                  # the filter does something
    for ns in (1, 2, 4):
        Yd = ddo.dd_chebyshev_filter(op, X, ns, m, a, b, a0)
        assert np.abs(Yd - Y).max() <= 1e-12 * np.abs(Y).max(), ns
    Y32 = ddo.dd_chebyshev_filter(op, X, 2, m, a, b, a0, fp32_payload=True)
    dev = np.abs(Y32 - Y).max() / np.abs(Y).max()
    assert 1e-10 < dev < 1e-4                                           # FP32 roundoff per step, not FP64, not O(1)
    assert np.array_equal(ddo.dd_chebyshev_filter(op, X, 1, m, a, b, a0, fp32_payload=True), ddo.dd_chebyshev_filter(op, X, 1, m, a, b, a0))


def plane_local_sets(mesh, rng, nsets_per_plane=2, planes=None):
    """Closed constraint sets whose nodes all lie in ONE node plane each (so that no set straddles a z-cut): per chosen
    plane a master-less set (a "hole" pinned to zero) and sets with 2-4 masters and 1-3 slaves."""
    from oracle import constraints_oracle as co
    ndx, ndy, ndz = mesh.nd
    plane = ndx * ndy
    sets = []
    for iz in (range(ndz) if planes is None else planes):
        nodes = iz * plane + rng.permutation(plane)
        k = 0
        sets.append(co.ConstraintSet([], nodes[k:k + 2], np.zeros((2, 0)), None)); k += 2
        for _ in range(nsets_per_plane):
            nm, ns = int(rng.integers(2, 5)), int(rng.integers(1, 4))
            sets.append(co.ConstraintSet(nodes[k:k + nm], nodes[k + nm:k + nm + ns], rng.uniform(-1, 1, (ns, nm)), None))
            k += nm + ns
    return sets


@pytest.mark.parametrize("bc", ["periodic", "dirichlet"])
def test_equation_17_in_full_constraints_inside_the_decomposed_apply(bc):
    """sum_t P^T C_t^T A_t C_t P U = C^T A C U for sets that live inside node planes -- the cut planes included, whose
    sets belong to two tasks -- and a set that straddles a cut is refused."""
    from oracle import constraints_oracle as co
    p, nc = 2, (2, 3, 4)
    mesh = orc.Mesh(nc, p, bc, (0.0, 0.0, 0.0), (1.0, 1.2, 2.0))
    op = orc.Operator(mesh, 0.7)
    rng = np.random.default_rng(17)
    sets = plane_local_sets(mesh, rng)
    X = rng.uniform(-1, 1, (mesh.ndof, 3))
    Y = co.distribute_transpose(sets, op.apply(co.distribute(sets, X, homogeneous=True)))
    assert np.abs(Y - op.apply(X)).max() > 1e-3 * np.abs(Y).max()          # the constraints matter
    for ns in (1, 2, 4):
        Yd = ddo.dd_constrained_apply(op, X, ns, sets)
        assert np.abs(Yd - Y).max() <= 1e-13 * np.abs(Y).max(), ns
    # a set that straddles a cut: master in plane 5, slave in plane 1, both nodes otherwise unconstrained
    plane = mesh.nd[0] * mesh.nd[1]
    used = set(int(v) for I in sets for v in np.concatenate([I.masters, I.slaves]))
    free5 = next(r for r in range(5 * plane, 6 * plane) if r not in used)
    free1 = next(r for r in range(plane, 2 * plane) if r not in used)
    with pytest.raises(ValueError):
        ddo.dd_constrained_apply(op, X, 4, sets + [co.ConstraintSet([free5], [free1], [[0.5]], None)])
