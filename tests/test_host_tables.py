"""Host logic of S0 without a GPU: the 1-D tables and the geometric factors that `fe_mf_create` computes in
paper_2208_07129_b200/csrc/fe_tables.h (long double, Newton-polished roots) are dumped by a small host-only C++ program and
compared with the oracle's (written independently in numpy long double) and with what the mathematics fixes."""
import os
import subprocess

import numpy as np
import pytest

from oracle import fe_oracle as orc

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def dumper(tmp_path_factory):
    exe = str(tmp_path_factory.mktemp("host") / "dump_tables")
    subprocess.run(["g++", "-O1", "-std=c++17", "-o", exe, os.path.join(ROOT, "tests", "host", "dump_tables.cpp")], check=True)
    return exe


def dump(exe, p):
    out = subprocess.run([exe, str(p)], capture_output=True, text=True, check=True).stdout
    d = {}
    for line in out.splitlines():
        k, *v = line.split()
        d[k] = np.array([float(x) for x in v])
    return d


@pytest.mark.parametrize("p", [1, 2, 3, 4, 5, 6, 7, 8])
def test_tables_match_the_oracle_and_their_identities(dumper, p):
    d = dump(dumper, p)
    n = p + 1
    xi, xq, w, N1, D1 = orc.tables_1d(p)
    Dt = orc.collocation_derivative_1d(p)
    assert np.abs(d["xi"] - xi).max() <= 4e-16 and np.abs(d["xq"] - xq).max() <= 4e-16 and np.abs(d["w"] - w).max() <= 4e-16
    N = d["N"].reshape(n, n); D = d["Dt"].reshape(n, n)
    assert np.abs(N - N1).max() <= 2e-15                                 # N[q][i] = l_i(xq_q)
    assert np.abs(D - Dt).max() <= 2e-13 * max(1.0, np.abs(Dt).max())    # D~[q][r] = l~_r'(xq_q)
    assert np.abs(D @ N - D1).max() <= 1e-12 * max(1.0, np.abs(D1).max())   # D = D~ N
    assert np.abs(N.sum(1) - 1).max() <= 1e-14 and np.abs(D.sum(1)).max() <= 1e-12
    assert abs(w.sum() - 2) <= 1e-15
    # the even-odd kernels rely on EXACT centro-(anti)symmetry of the uploaded tables (reading 14)
    assert np.array_equal(N, N[::-1, ::-1]) and np.array_equal(D, -D[::-1, ::-1])
    assert np.array_equal(d["xq"], -d["xq"][::-1]) and np.array_equal(d["w"], d["w"][::-1])


def test_trilinear_jacobian_and_metric(dumper):
    """J = dx/dxi of the trilinear map and G = J^-1 J^-T det J at one point of a distorted cell."""
    d = dump(dumper, 2)
    v = np.array([[0, 0, 0], [1.1, 0.05, -0.02], [0.03, 0.9, 0.04], [1.0, 1.05, 0.1],
                  [-0.05, 0.02, 1.2], [1.08, 0.0, 1.1], [0.1, 1.0, 1.15], [1.2, 0.95, 1.3]])
    xi = np.array([[0.3, -0.55, 0.8]])
    _, J = orc.trilinear_map(v, xi)
    J = J[0]
    assert np.abs(d["J"].reshape(3, 3) - J).max() <= 1e-15
    det = np.linalg.det(J)
    Ginv = np.linalg.inv(J) @ np.linalg.inv(J).T * det
    m = d["metric"]
    assert m[0] == 1.0
    ref = np.array([Ginv[0, 0], Ginv[0, 1], Ginv[0, 2], Ginv[1, 1], Ginv[1, 2], Ginv[2, 2], det])
    assert np.abs(m[1:] - ref).max() <= 1e-14 * np.abs(ref).max()
