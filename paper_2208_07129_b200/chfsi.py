"""ctypes binding of include/fe_chfsi.h (argument marshalling only): Chebyshev filtered subspace iteration around a
`binding.FeMf` operator.  Same names as the C entry points minus the prefix."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import binding
from .binding import FE_MF_OK, FeMfError, _check_tensor, _stream_ptr

LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "csrc", "libfe_chfsi.so")
_PD = C.POINTER(C.c_double)

SYMBOLS = {
    "fe_chfsi_create": (C.c_int, [C.POINTER(C.c_void_p), C.c_void_p, C.c_int]),
    "fe_chfsi_destroy": (None, [C.c_void_p]),
    "fe_chfsi_last_error": (C.c_char_p, [C.c_void_p]),
    "fe_chfsi_lanczos_bound": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, _PD, C.c_void_p]),
    "fe_chfsi_orthonormalize": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "fe_chfsi_rayleigh_ritz": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, _PD, _PD, C.c_void_p]),
    "fe_chfsi_iterate": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_double, _PD, _PD,
                                   C.c_void_p]),
    "fe_chfsi_solve": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                 C.c_double, C.c_int, _PD, _PD, C.POINTER(C.c_int), C.c_void_p]),
    "fe_chfsi_last_timings": (C.c_int, [C.c_void_p, _PD]),
}

_lib = None


def lib():
    global _lib
    if _lib is None:
        binding.lib()                      # libfe_mf.so first: libfe_chfsi.so links it
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2208_07129_b200.build` "
                               "(there is no CPU fallback)")
        l = C.CDLL(LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(l, name)
            fn.restype, fn.argtypes = res, args
        _lib = l
    return _lib


class Chfsi:
    def __init__(self, op: "binding.FeMf", nvec: int):
        self._l = lib()
        self._h = C.c_void_p()
        self.op, self.nvec = op, int(nvec)
        rc = self._l.fe_chfsi_create(C.byref(self._h), op._ctx, int(nvec))
        if rc != FE_MF_OK:
            raise FeMfError(rc, self._l.fe_chfsi_last_error(None).decode())

    def _raise(self, rc: int):
        if rc != FE_MF_OK:
            raise FeMfError(rc, self._l.fe_chfsi_last_error(self._h).decode())

    def lanczos_bound(self, v0, k: int = 10, stream=None) -> float:
        _check_tensor(v0, self.op.ndofs, 1, "v0")
        out = C.c_double()
        self._raise(self._l.fe_chfsi_lanczos_bound(self._h, v0.data_ptr(), int(k), C.byref(out), _stream_ptr(stream)))
        return out.value

    def orthonormalize(self, X, stream=None):
        _check_tensor(X, self.op.ndofs, self.nvec, "X")
        self._raise(self._l.fe_chfsi_orthonormalize(self._h, X.data_ptr(), _stream_ptr(stream)))

    def rayleigh_ritz(self, X, U, stream=None):
        _check_tensor(X, self.op.ndofs, self.nvec, "X"); _check_tensor(U, self.op.ndofs, self.nvec, "U")
        lam, res = np.empty(self.nvec), np.empty(self.nvec)
        self._raise(self._l.fe_chfsi_rayleigh_ritz(self._h, X.data_ptr(), U.data_ptr(), lam.ctypes.data_as(_PD),
                                                   res.ctypes.data_as(_PD), _stream_ptr(stream)))
        return lam, res

    def iterate(self, U, m: int, lam_max: float, lam_u: float, lam_min: float, stream=None):
        _check_tensor(U, self.op.ndofs, self.nvec, "U")
        lam, res = np.empty(self.nvec), np.empty(self.nvec)
        self._raise(self._l.fe_chfsi_iterate(self._h, U.data_ptr(), int(m), float(lam_max), float(lam_u),
                                             float(lam_min), lam.ctypes.data_as(_PD), res.ctypes.data_as(_PD),
                                             _stream_ptr(stream)))
        return lam, res

    def solve(self, U, n_wanted: int, m: int, lam_max: float, lam_u: float, lam_min: float, tau: float,
              max_iter: int = 50, stream=None):
        _check_tensor(U, self.op.ndofs, self.nvec, "U")
        lam, res = np.empty(self.nvec), np.empty(self.nvec)
        it = C.c_int()
        self._raise(self._l.fe_chfsi_solve(self._h, U.data_ptr(), int(n_wanted), int(m), float(lam_max), float(lam_u),
                                           float(lam_min), float(tau), int(max_iter), lam.ctypes.data_as(_PD),
                                           res.ctypes.data_as(_PD), C.byref(it), _stream_ptr(stream)))
        return lam, res, it.value

    def last_timings(self) -> dict:
        ms = (C.c_double * 6)()
        self._raise(self._l.fe_chfsi_last_timings(self._h, ms))
        return dict(zip(("filter", "orthonormalize", "operator", "gemm", "syevd", "residual"), list(ms)))

    def destroy(self):
        if getattr(self, "_h", None) and self._h.value:
            self._l.fe_chfsi_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
