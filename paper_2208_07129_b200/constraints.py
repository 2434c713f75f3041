"""ctypes binding of include/fe_constraints.h: the constraint matrices C, C^T as
sets of (masters, slaves, W_I, b_I).  Argument marshalling only; the arithmetic is in libfe_mf.so."""
from __future__ import annotations

import ctypes as C
from typing import Optional, Sequence

import numpy as np

from . import binding

_PLL = C.POINTER(C.c_longlong)
_PD = C.POINTER(C.c_double)
# every symbol include/fe_constraints.h declares: name -> (restype, argtypes)
SYMBOLS = {
    "fe_constraints_create": (C.c_int, [C.POINTER(C.c_void_p), C.c_longlong, C.c_int, _PLL, _PLL, _PLL, _PLL, _PD, _PD, C.c_int]),
    "fe_constraints_distribute": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p]),
    "fe_constraints_distribute_transpose": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]),
    "fe_constraints_counts": (C.c_int, [C.c_void_p, C.POINTER(C.c_int), _PLL, _PLL]),
    "fe_constraints_last_error": (C.c_char_p, [C.c_void_p]),
    "fe_constraints_destroy": (None, [C.c_void_p]),
}
_declared = False


def lib():
    """libfe_mf.so with the fe_constraints_* prototypes declared (built on demand; fails loudly without nvcc)."""
    global _declared
    L = binding.lib()
    if not _declared:
        for name, (res, args) in SYMBOLS.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _declared = True
    return L


def _ll(a):
    a = np.ascontiguousarray(a, dtype=np.int64).reshape(-1)
    return a, a.ctypes.data_as(_PLL)


class Constraints:
    """The constraint sets of one task.  `sets`: sequence of (masters, slaves, W, b) with W [ns][nm] and b [ns] or None."""

    def __init__(self, ndof: int, sets: Sequence, device: int = 0):
        L = lib()
        m_ptr, s_ptr = [0], [0]
        masters, slaves, weights, inhomog = [], [], [], []
        for (ms, sl, W, b) in sets:
            ms = np.asarray(ms, dtype=np.int64).reshape(-1)
            sl = np.asarray(sl, dtype=np.int64).reshape(-1)
            W = np.asarray(W, dtype=np.float64)
            if W.size != len(sl) * len(ms):
                raise ValueError("W must be [len(slaves)][len(masters)]")
            b = np.zeros(len(sl)) if b is None else np.asarray(b, dtype=np.float64).reshape(-1)
            if len(b) != len(sl):
                raise ValueError("one inhomogeneity per slave")
            masters.append(ms); slaves.append(sl); weights.append(W.reshape(-1)); inhomog.append(b)
            m_ptr.append(m_ptr[-1] + len(ms)); s_ptr.append(s_ptr[-1] + len(sl))
        cat = lambda parts, dt: np.concatenate(parts).astype(dt) if parts else np.zeros(0, dtype=dt)   # noqa: E731
        self._keep = [_ll(m_ptr), _ll(cat(masters, np.int64)), _ll(s_ptr), _ll(cat(slaves, np.int64))]
        w = np.ascontiguousarray(cat(weights, np.float64)); bb = np.ascontiguousarray(cat(inhomog, np.float64))
        self._h = C.c_void_p()
        rc = L.fe_constraints_create(C.byref(self._h), int(ndof), len(sets), self._keep[0][1], self._keep[1][1],
                                     self._keep[2][1], self._keep[3][1], w.ctypes.data_as(_PD), bb.ctypes.data_as(_PD),
                                     int(device))
        if rc != binding.FE_MF_OK:
            self._h = C.c_void_p()
            raise binding.FeMfError(rc, L.fe_constraints_last_error(None).decode())
        self.ndof, self.device = int(ndof), int(device)

    def _check(self, X, nvec):
        import torch
        assert isinstance(X, torch.Tensor) and X.is_cuda and X.dtype == torch.float64 and X.is_contiguous()
        assert X.numel() == self.ndof * nvec and X.device.index == self.device

    def _raise(self, rc):
        raise binding.FeMfError(rc, lib().fe_constraints_last_error(self._h).decode())

    def distribute(self, U, nvec: int, homogeneous: bool = False, stream=None):
        """U <- C U (+ b unless homogeneous), in place (fe_constraints_distribute)."""
        self._check(U, nvec)
        rc = lib().fe_constraints_distribute(self._h, U.data_ptr(), int(nvec), 1 if homogeneous else 0, binding._stream_ptr(stream))
        if rc != binding.FE_MF_OK:
            self._raise(rc)
        return U

    def distribute_transpose(self, V, nvec: int, stream=None):
        """V <- C^T V, in place (fe_constraints_distribute_transpose)."""
        self._check(V, nvec)
        rc = lib().fe_constraints_distribute_transpose(self._h, V.data_ptr(), int(nvec), binding._stream_ptr(stream))
        if rc != binding.FE_MF_OK:
            self._raise(rc)
        return V

    def counts(self):
        n, nm, ns = C.c_int(), C.c_longlong(), C.c_longlong()
        lib().fe_constraints_counts(self._h, C.byref(n), C.byref(nm), C.byref(ns))
        return n.value, nm.value, ns.value

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().fe_constraints_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def constrained_apply(op, cons: Constraints, X, Y, nvec: int, work: Optional[object] = None, stream=None):
    """Y = C^T A C X (Eq. 17, one task): X is left untouched -- C acts on a copy (`work`, same shape; the
    copy is enqueued on torch's current stream, so `stream`, if given, must be that stream)."""
    if work is None:
        work = X.new_empty(X.shape)
    work.copy_(X)
    cons.distribute(work, nvec, homogeneous=True, stream=stream)
    op.apply(work, Y, nvec, stream)
    cons.distribute_transpose(Y, nvec, stream=stream)
    return Y
