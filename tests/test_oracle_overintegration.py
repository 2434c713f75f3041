"""Pins of the oracle with n_q = n_p + 2 Gauss points per direction.
No GPU."""
import numpy as np
import pytest

import importlib.util
import os

from oracle import fe_oracle as orc
from paper_2208_07129_b200 import inputs

_spec = importlib.util.spec_from_file_location("_oracle_pins", os.path.join(os.path.dirname(__file__), "test_oracle_pins.py"))
_pins = importlib.util.module_from_spec(_spec)
_spec.loader.exec_module(_pins)
_brute_force_cell = _pins._brute_force_cell      # the long-double (I, J, Q) loops with their own basis and Jacobian


@pytest.mark.parametrize("p", [1, 2, 3])
def test_distorted_cell_brute_force_with_more_points(p):
    """Long-double loops over (I, J, Q) with an independent basis and Jacobian evaluation, n_q = p + 3."""
    rng = np.random.default_rng(17 + p)
    verts = np.array([[(v & 1), (v >> 1) & 1, (v >> 2) & 1] for v in range(8)], dtype=float) * [1.0, 1.4, 0.8]
    verts += rng.uniform(-0.12, 0.12, verts.shape)
    nq = p + 3
    Nf, Df, W = orc.tables_3d(p, nq)
    assert Nf.shape == (nq ** 3, (p + 1) ** 3) and Df.shape == (3, nq ** 3, (p + 1) ** 3) and W.shape == (nq ** 3,)
    qpts, _ = orc.reference_points_3d(p, nq)
    G, g = orc.geometric_factors(verts, qpts, W, 0.9)
    A = orc.element_matrix(Nf, Df, G, g)
    ref = _brute_force_cell(p, verts, 0.9, nq)
    assert np.abs(A - np.asarray(ref, dtype=np.float64)).max() <= 1e-13 * float(np.abs(ref).max())


@pytest.mark.parametrize("p", [1, 2, 4])
@pytest.mark.parametrize("bc", ["periodic", "dirichlet"])
def test_affine_cells_are_already_exact(p, bc):
    """On affine cells the integrands are polynomials of degree 2p per direction: the n_p-point rule (exact to 2p+1) and
    the (n_p+2)-point rule give the same operator -- uniform box and sheared parallelepipeds."""
    nc = (2, 3, 2)
    X = inputs.multivector(3, orc.Mesh(nc, p, bc).ndof, 3)
    m0 = orc.Mesh(nc, p, bc, (0, 0, 0), (1.0, 2.0, 0.7))
    a, b = orc.Operator(m0, 0.8).apply(X), orc.Operator(m0, 0.8, nq=p + 3).apply(X)
    assert np.abs(a - b).max() <= 1e-12 * np.abs(a).max()
    if bc == "dirichlet":
        v = inputs.uniform_vertices(nc, (0, 0, 0), (1, 1, 1)) @ np.array([[1.0, 0.3, 0.1], [0.0, 1.1, 0.2], [0.0, 0.0, 0.9]]).T
        m1 = orc.Mesh(nc, p, bc, vertices=v)
        a, b = orc.Operator(m1, 0.8).apply(X), orc.Operator(m1, 0.8, nq=p + 3).apply(X)
        assert np.abs(a - b).max() <= 1e-12 * np.abs(a).max()


def test_trilinear_cells_differ_and_converge():
    """On a perturbed mesh the metric is rational: n_p and n_p + 2 points differ visibly, n_p + 2 and n_p + 4 much
    less (the quadrature error of the Gauss rule falls with the number of points); invariants hold for every rule."""
    p, nc = 3, (3, 2, 3)
    v = inputs.perturbed_vertices(nc, (0, 0, 0), (1.0, 0.8, 1.2), 0.15, 99)
    mesh = orc.Mesh(nc, p, "periodic", (0, 0, 0), (1.0, 0.8, 1.2), vertices=v)
    X = inputs.multivector(5, mesh.ndof, 2)
    Y = [orc.Operator(mesh, 0.7, nq=p + 1 + 2 * k).apply(X) for k in range(3)]
    d01, d12 = np.abs(Y[0] - Y[1]).max(), np.abs(Y[1] - Y[2]).max()
    scale = np.abs(Y[2]).max()
    assert d01 > 1e-7 * scale and d12 < 0.05 * d01
    one = np.ones((mesh.ndof, 1))
    for nq in (p + 1, p + 3):
        assert np.abs(orc.Operator(mesh, 1.0, ck=1.0, cm=0.0, nq=nq).apply(one)).max() < 1e-12     # K 1 = 0
        assert abs(float((one.T @ orc.Operator(mesh, 1.0, ck=0.0, cm=1.0, nq=nq).apply(one)).item()) - 0.96) < 1e-13   # |Omega|
        op = orc.Operator(mesh, 0.7, nq=nq)
        u, w = inputs.multivector(11, mesh.ndof, 1), inputs.multivector(12, mesh.ndof, 1)
        assert abs(np.sum(u * op.apply(w)) - np.sum(w * op.apply(u))) <= 1e-12 * abs(np.sum(u * op.apply(w)))


def test_kappa_array_has_one_value_per_point_of_the_rule():
    """kappa at n_q^3 points: the bilinear-kappa moments of tests/test_oracle_mass_scaled.py with n_q = p + 3."""
    a, b, c, p = 1.0, 2.0, 1.5, 2
    m = orc.Mesh((3, 2, 2), p, "natural", (0, 0, 0), (a, b, c))
    xq = orc.quadrature_point_coordinates(m, p + 3)
    assert xq.shape == (12, (p + 3) ** 3, 3)
    kap = 1 + 2 * xq[..., 0] + 3 * xq[..., 1] - xq[..., 2] + xq[..., 0] * xq[..., 1]
    r = orc.Operator(m, 0.0, ck=0.0, cm=1.0, kappa=kap, nq=p + 3).apply(np.ones(m.ndof))
    V = a * b * c
    assert abs(r.sum() - V * (1 + a + 1.5 * b - 0.5 * c + a * b / 4)) < 1e-13 * r.sum()
    X = m.node_coordinates()
    assert abs(X[:, 2] @ r - V * (c / 2 + a * c / 2 + 3 * b * c / 4 - c * c / 3 + a * b * c / 8)) < 1e-12
