"""No-GPU checks of the boundary: the C-ABI library builds, loads, and exports every symbol that
include/fe_mf.h declares; the binding's symbol table matches the header; the product path fails
loudly without a device (no CPU fallback)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_symbols(header="fe_mf.h"):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(fe_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def built_lib():
    from paper_2208_07129_b200 import build
    return build.build()


def test_header_declares_the_north_star_entry_points():
    syms = header_symbols()
    for name in ("fe_mf_create", "fe_mf_apply", "fe_cheb_filter", "fe_mf_destroy", "fe_mf_ndofs", "fe_mf_last_error"):
        assert name in syms


def test_library_exports_every_declared_symbol(built_lib):
    lib = ctypes.CDLL(built_lib)
    for name in header_symbols():
        assert hasattr(lib, name), name


def test_binding_table_matches_header(built_lib):
    from paper_2208_07129_b200 import binding
    assert sorted(binding.SYMBOLS) == header_symbols()
    binding.lib()


def test_chfsi_library_exports_every_declared_symbol(built_lib):
    """include/fe_chfsi.h: libfe_chfsi.so builds, loads and exports what the header declares;
    the binding's table matches."""
    from paper_2208_07129_b200 import build, chfsi
    path = build.build_chfsi()
    ctypes.CDLL(built_lib, mode=ctypes.RTLD_GLOBAL)
    lib = ctypes.CDLL(path)
    syms = [s for s in header_symbols("fe_chfsi.h") if s.startswith("fe_chfsi_")]
    assert "fe_chfsi_solve" in syms and "fe_chfsi_iterate" in syms
    for name in syms:
        assert hasattr(lib, name), name
    assert sorted(chfsi.SYMBOLS) == syms
    from paper_2208_07129_b200 import binding
    assert chfsi.lib().fe_chfsi_solve(None, None, 1, 1, 1.0, 0.5, 0.0, 1e-3, 1, None, None, None, None) == binding.FE_MF_EINVAL


def test_no_cpu_fallback(built_lib):
    """Without a CUDA device fe_mf_create must fail with a CUDA error, not compute on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2208_07129_b200 import binding
    with pytest.raises(binding.FeMfError) as e:
        binding.FeMf((2, 2, 2), 2, 1.0, binding.FE_BC_PERIODIC)
    assert e.value.code == binding.FE_MF_ECUDA


def test_argument_validation_without_gpu(built_lib):
    from paper_2208_07129_b200 import binding
    l = binding.lib()
    assert l.fe_mf_ndofs(None) == -1
    assert l.fe_mf_apply(None, None, None, 1, None) == binding.FE_MF_EINVAL
    ctx = ctypes.c_void_p()
    lo = (ctypes.c_double * 3)(0, 0, 0); hi = (ctypes.c_double * 3)(1, 1, 1)
    assert l.fe_mf_create(ctypes.byref(ctx), 2, 2, 2, 0, 1.0, 0, 0, lo, hi, None, 0) == binding.FE_MF_EINVAL
    assert b"p must be" in l.fe_mf_last_error(None)
    assert l.fe_mf_create(None, 2, 2, 2, 2, 1.0, 0, 0, lo, hi, None, 0) == binding.FE_MF_EINVAL


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2208_07129_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".inl")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
    orc = open(os.path.join(ROOT, "oracle", "fe_oracle.py")).read()
    assert "paper_2208_07129_b200" not in orc.replace("`paper_2208_07129_b200/csrc`", "")


def test_roofline_counts():
    """The work model of paper_2208_07129_b200/roofline.py (pure counting): the even-odd count per DoF*vector quoted in
    SURVEY.md 8(d) / DESIGN.md section 6, the rectangular count of the n_q != n_p rule reducing to it at n_q = n_p, and the
    non-even-odd total 24 n^4 + 16 n^3 flops per cell and vector of PAPER.md:203."""
    from paper_2208_07129_b200 import roofline
    assert abs(roofline.work_per_dof_vec(6, True)[0] - 107.07) < 0.01       # Cartesian-diagonal metric, p = 6
    assert abs(roofline.work_per_dof_vec(6, False)[0] - 116.6) < 0.01
    assert abs(roofline.work_per_dof_vec(8, False)[0] - 122.45) < 0.01
    for p in range(1, 9):
        for diag in (True, False):
            a = roofline.work_per_dof_vec(p, diag)
            b = roofline.work_per_dof_vec_oi(p, p + 1, diag)
            assert abs(a[0] - b[0]) < 1e-12 and abs(a[1] - b[1]) < 1e-12
        n = p + 1
        fma, other = roofline.fp64_instr_per_cell_vec(p, False, even_odd=False)
        assert 2 * fma + other == 24 * n ** 4 + 16 * n ** 3
    assert roofline.work_per_dof_vec_oi(8, 11, False)[0] > 1.7 * roofline.work_per_dof_vec(8, False)[0]
    assert roofline.bytes_per_dof_vec(6, False, 16) == 16.0 and roofline.bytes_per_dof_vec(6, False, 16, chebyshev=True) == 24.0


def test_constraints_header_symbols_and_validation_without_gpu(built_lib):
    """include/fe_constraints.h: libfe_mf.so exports what the header declares, the
    binding's table matches, the host-side validation of the sets (closed sets, index ranges, offsets) answers EINVAL
    before any device is touched, and valid sets without a device fail with ECUDA (no CPU fallback)."""
    import torch
    from paper_2208_07129_b200 import binding, constraints
    lib = ctypes.CDLL(built_lib)
    syms = header_symbols("fe_constraints.h")
    assert "fe_constraints_create" in syms and "fe_constraints_distribute_transpose" in syms
    for name in syms:
        assert hasattr(lib, name), name
    assert sorted(constraints.SYMBOLS) == syms
    L = constraints.lib()
    LL = ctypes.c_longlong

    def create(ndof, m_ptr, masters, s_ptr, slaves, weights):
        h = ctypes.c_void_p()
        arr = lambda v: (LL * max(len(v), 1))(*v)      # noqa: E731
        w = (ctypes.c_double * max(len(weights), 1))(*weights)
        rc = L.fe_constraints_create(ctypes.byref(h), ndof, len(m_ptr) - 1, arr(m_ptr), arr(masters), arr(s_ptr), arr(slaves),
                                     w, None, 0)
        return rc, h, L.fe_constraints_last_error(None)

    rc, h, msg = create(5, [0, 1, 2], [1, 2], [0, 1, 2], [2, 3], [1.0, 1.0])          # slave 2 is a master of set 1
    assert rc == binding.FE_MF_EINVAL and b"not closed" in msg and not h.value
    rc, h, msg = create(5, [0, 1, 2], [1, 0], [0, 1, 2], [2, 2], [1.0, 1.0])          # slave 2 twice
    assert rc == binding.FE_MF_EINVAL and b"two sets" in msg
    rc, h, msg = create(5, [0, 1], [7], [0, 1], [2], [1.0])                           # master out of range
    assert rc == binding.FE_MF_EINVAL and b"out of range" in msg
    rc, h, msg = create(5, [0, 1], [1], [0, 1], [-1], [1.0])
    assert rc == binding.FE_MF_EINVAL and b"out of range" in msg
    rc, h, msg = create(5, [1, 1], [1], [0, 1], [2], [])                              # offsets must start at 0
    assert rc == binding.FE_MF_EINVAL
    rc, h, msg = create(0, [0], [], [0], [], [])
    assert rc == binding.FE_MF_EINVAL
    assert L.fe_constraints_distribute(None, None, 1, 0, None) == binding.FE_MF_EINVAL
    assert L.fe_constraints_distribute_transpose(None, None, 1, None) == binding.FE_MF_EINVAL
    assert L.fe_constraints_counts(None, None, None, None) == binding.FE_MF_EINVAL
    L.fe_constraints_destroy(None)
    if not torch.cuda.is_available():
        with pytest.raises(binding.FeMfError) as e:
            constraints.Constraints(5, [([1], [2], [[1.0]], None)])
        assert e.value.code == binding.FE_MF_ECUDA
