"""Thin ctypes binding of include/fe_mf.h -- argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/libfe_mf.so.  PyTorch is used by callers
for device memory and streams; this module only passes `data_ptr()`s and the current stream.
There is no fallback: if the library is missing or fails to load, `lib()` raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "csrc", "libfe_mf.so")

FE_MF_OK, FE_MF_EINVAL, FE_MF_ENOMEM, FE_MF_ECUDA, FE_MF_EUNSUPPORTED = 0, 1, 2, 3, 4
FE_BC_PERIODIC, FE_BC_DIRICHLET = 0, 1
FE_GEOM_AFFINE, FE_GEOM_QPOINT = 0, 1

# every symbol include/fe_mf.h declares: name -> (restype, argtypes)
_D = C.c_double
_PD = C.POINTER(C.c_double)
SYMBOLS = {
    "fe_mf_create": (C.c_int, [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, C.c_int, _D, C.c_int, C.c_int,
                               _PD, _PD, C.c_void_p, C.c_int]),
    "fe_mf_create_slab": (C.c_int, [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, C.c_int, _D, C.c_int, C.c_int,
                                    _PD, _PD, C.c_void_p, C.c_int, C.c_int]),
    "fe_mf_halo_add": (C.c_int, [C.c_void_p, C.c_void_p, C.c_longlong, C.c_void_p]),
    "fe_mf_axpby": (C.c_int, [C.c_void_p, C.c_void_p, _D, _D, C.c_longlong, C.c_void_p]),
    "fe_mf_halo_pack_f32": (C.c_int, [C.c_void_p, C.c_void_p, C.c_longlong, C.c_void_p]),
    "fe_mf_halo_unpack_f32": (C.c_int, [C.c_void_p, C.c_void_p, C.c_longlong, C.c_int, C.c_void_p]),
    "fe_mf_ndofs": (C.c_longlong, [C.c_void_p]),
    "fe_mf_apply": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]),
    "fe_mf_apply_bcv": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p]),
    "fe_mf_apply_axpby": (C.c_int, [C.c_void_p, _D, C.c_void_p, _D, _D, C.c_void_p, C.c_int, C.c_void_p]),
    "fe_mf_accumulate": (C.c_int, [C.c_void_p, _D, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]),
    "fe_cheb_filter": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, _D, _D, _D, C.c_void_p]),
    "fe_mf_apply_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]),
    "fe_fill_uniform": (C.c_int, [C.c_void_p, C.c_longlong, C.c_ulonglong, C.c_longlong, C.c_void_p]),
    "fe_probe_peaks": (C.c_int, [_PD, _PD, C.c_int]),
    "fe_mf_batch_width": (C.c_int, [C.c_void_p, C.c_int]),
    "fe_mf_shape": (C.c_int, [C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int)]),
    "fe_mf_kernel_name": (C.c_char_p, [C.c_void_p, C.c_int]),
    "fe_mf_last_launch_count": (C.c_int, [C.c_void_p]),
    "fe_mf_set_variant": (C.c_int, [C.c_void_p, C.c_int]),
    "fe_mf_set_kappa": (C.c_int, [C.c_void_p, _PD]),
    "fe_mf_set_quadrature": (C.c_int, [C.c_void_p, C.c_int]),
    "fe_mf_set_mass_scaling": (C.c_int, [C.c_void_p, C.c_int]),
    "fe_mf_mass_diagonal": (C.c_int, [C.c_void_p, _PD]),
    "fe_mf_last_error": (C.c_char_p, [C.c_void_p]),
    "fe_mf_destroy": (None, [C.c_void_p]),
}

_lib = None


class FeMfError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"fe_mf error {code}: {msg}")
        self.code = code


def lib() -> C.CDLL:
    """Load libfe_mf.so (built by `python -m paper_2208_07129_b200.build`).  Fails loudly."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2208_07129_b200.build` "
                               "(there is no CPU fallback)")
        l = C.CDLL(LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(l, name)
            fn.restype, fn.argtypes = res, args
        _lib = l
    return _lib


def _stream_ptr(stream) -> Optional[int]:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if hasattr(stream, "cuda_stream"):
        return stream.cuda_stream
    return int(stream)


def _check_tensor(t, ndof: int, nvec: int, name: str):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError(f"{name} must be a contiguous float64 CUDA tensor")
    if t.numel() != ndof * nvec:
        raise ValueError(f"{name} has {t.numel()} elements, expected {ndof}*{nvec}")


class FeMf:
    """fe_mf_ctx owner.  Methods carry the same names as the C entry points (minus the prefix)."""

    def __init__(self, ncells: Sequence[int], p: int, sigma: float, bc: int, geom: int = FE_GEOM_AFFINE,
                 box_lo=(0.0, 0.0, 0.0), box_hi=(1.0, 1.0, 1.0), vertices: Optional[np.ndarray] = None,
                 device: int = 0, z_open: Optional[int] = None):
        """z_open: None = a whole mesh (fe_mf_create); 0..3 = one z-slab of a decomposed mesh (fe_mf_create_slab)."""
        self._l = lib()
        self._ctx = C.c_void_p()
        lo = (C.c_double * 3)(*[float(v) for v in box_lo])
        hi = (C.c_double * 3)(*[float(v) for v in box_hi])
        vptr = None
        if vertices is not None:
            v = np.ascontiguousarray(vertices, dtype=np.float64)
            if v.shape != (ncells[2] + 1, ncells[1] + 1, ncells[0] + 1, 3):
                raise ValueError("vertices must have shape (ncz+1, ncy+1, ncx+1, 3)")
            self._verts = v
            vptr = v.ctypes.data_as(C.c_void_p)
        if z_open is None:
            rc = self._l.fe_mf_create(C.byref(self._ctx), int(ncells[0]), int(ncells[1]), int(ncells[2]), int(p),
                                      float(sigma), int(bc), int(geom), lo, hi, vptr, int(device))
        else:
            rc = self._l.fe_mf_create_slab(C.byref(self._ctx), int(ncells[0]), int(ncells[1]), int(ncells[2]), int(p),
                                           float(sigma), int(bc), int(geom), lo, hi, vptr, int(z_open), int(device))
        if rc != FE_MF_OK:
            raise FeMfError(rc, self._l.fe_mf_last_error(None).decode())
        self.ndofs = int(self._l.fe_mf_ndofs(self._ctx))
        self.p, self.device = int(p), int(device)
        self.ncells = tuple(int(c) for c in ncells)
        self.nq = int(p) + 1

    @classmethod
    def from_workload(cls, w, device: int = 0) -> "FeMf":
        from . import inputs
        return cls(w.ncells, w.p, w.sigma, w.bc, w.geom, w.box_lo, w.box_hi, inputs.workload_vertices(w), device)

    def _raise(self, rc: int):
        if rc != FE_MF_OK:
            raise FeMfError(rc, self._l.fe_mf_last_error(self._ctx).decode())

    def apply(self, X, Y, nvec: int, stream=None):
        _check_tensor(X, self.ndofs, nvec, "X"); _check_tensor(Y, self.ndofs, nvec, "Y")
        self._raise(self._l.fe_mf_apply(self._ctx, X.data_ptr(), Y.data_ptr(), int(nvec), _stream_ptr(stream)))

    def apply_bcv(self, X, Y, b: int, nvec: int, stream=None):
        """The apply on the paper's BCV layout (fe_mf_apply_bcv): batches of b vectors, each a contiguous [ndofs][b] block."""
        _check_tensor(X, self.ndofs, nvec, "X"); _check_tensor(Y, self.ndofs, nvec, "Y")
        self._raise(self._l.fe_mf_apply_bcv(self._ctx, X.data_ptr(), Y.data_ptr(), int(b), int(nvec), _stream_ptr(stream)))

    def apply_axpby(self, alpha: float, W, beta: float, gamma: float, Z, nvec: int, stream=None):
        _check_tensor(W, self.ndofs, nvec, "W"); _check_tensor(Z, self.ndofs, nvec, "Z")
        self._raise(self._l.fe_mf_apply_axpby(self._ctx, float(alpha), W.data_ptr(), float(beta), float(gamma),
                                              Z.data_ptr(), int(nvec), _stream_ptr(stream)))

    def accumulate(self, alpha: float, W, Z, nvec: int, stream=None):
        _check_tensor(W, self.ndofs, nvec, "W"); _check_tensor(Z, self.ndofs, nvec, "Z")
        self._raise(self._l.fe_mf_accumulate(self._ctx, float(alpha), W.data_ptr(), Z.data_ptr(), int(nvec),
                                             _stream_ptr(stream)))

    def cheb_filter(self, X, Y, nvec: int, m: int, a: float, b: float, a0: float, stream=None):
        _check_tensor(X, self.ndofs, nvec, "X"); _check_tensor(Y, self.ndofs, nvec, "Y")
        self._raise(self._l.fe_cheb_filter(self._ctx, X.data_ptr(), Y.data_ptr(), int(nvec), int(m), float(a),
                                           float(b), float(a0), _stream_ptr(stream)))

    def apply_host(self, X_host, Y_host, nvec: int):
        """X_host / Y_host: CPU float64 tensors or numpy arrays (pinned recommended)."""
        def ptr(t):
            if isinstance(t, np.ndarray):
                assert t.dtype == np.float64 and t.flags.c_contiguous and t.size == self.ndofs * nvec
                return t.ctypes.data
            assert (not t.is_cuda) and t.is_contiguous() and t.numel() == self.ndofs * nvec
            return t.data_ptr()
        self._raise(self._l.fe_mf_apply_host(self._ctx, ptr(X_host), ptr(Y_host), int(nvec)))

    def batch_width(self, nvec: int) -> int:
        return int(self._l.fe_mf_batch_width(self._ctx, int(nvec)))

    def kernel_name(self, nvec: int) -> str:
        return self._l.fe_mf_kernel_name(self._ctx, int(nvec)).decode()

    def last_launch_count(self) -> int:
        return int(self._l.fe_mf_last_launch_count(self._ctx))

    def set_variant(self, variant: int):
        self._raise(self._l.fe_mf_set_variant(self._ctx, int(variant)))

    def set_kappa(self, kappa):
        """kappa at the quadrature points, host array [ncells][n^3] (or None: back to the constant sigma)."""
        if kappa is None:
            self._raise(self._l.fe_mf_set_kappa(self._ctx, None))
            return
        k = np.ascontiguousarray(kappa, dtype=np.float64)
        n3 = self.nq ** 3
        if k.size != self.ncells[0] * self.ncells[1] * self.ncells[2] * n3:
            raise ValueError("kappa must have ncells * (p+1)^3 entries")
        self._raise(self._l.fe_mf_set_kappa(self._ctx, k.ctypes.data_as(_PD)))

    def set_quadrature(self, nq: int):
        """nq Gauss points per direction (p + 1 = default); a kappa array set before is dropped."""
        self._raise(self._l.fe_mf_set_quadrature(self._ctx, int(nq)))
        self.nq = int(nq)

    def set_mass_scaling(self, on: bool):
        self._raise(self._l.fe_mf_set_mass_scaling(self._ctx, 1 if on else 0))

    def mass_diagonal(self) -> np.ndarray:
        out = np.empty(self.ndofs, dtype=np.float64)
        self._raise(self._l.fe_mf_mass_diagonal(self._ctx, out.ctypes.data_as(_PD)))
        return out

    def destroy(self):
        if getattr(self, "_ctx", None) and self._ctx.value:
            self._l.fe_mf_destroy(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def fill_uniform(out, seed: int, offset: int = 0, stream=None):
    """out (float64 CUDA tensor) <- u(seed, offset + k); bit-identical to inputs.uniform_pm1."""
    import torch
    assert isinstance(out, torch.Tensor) and out.is_cuda and out.dtype == torch.float64 and out.is_contiguous()
    rc = lib().fe_fill_uniform(out.data_ptr(), out.numel(), int(seed), int(offset), _stream_ptr(stream))
    if rc != FE_MF_OK:
        raise FeMfError(rc, "fe_fill_uniform failed")
    return out


def halo_add(dst, src, stream=None):
    """dst += src on the device (fe_mf_halo_add): the receiving side of the P^(t)T step of a decomposed apply."""
    import torch
    assert isinstance(dst, torch.Tensor) and dst.is_cuda and dst.dtype == torch.float64 and dst.is_contiguous()
    assert isinstance(src, torch.Tensor) and src.is_cuda and src.dtype == torch.float64 and src.is_contiguous()
    assert dst.numel() == src.numel()
    rc = lib().fe_mf_halo_add(dst.data_ptr(), src.data_ptr(), dst.numel(), _stream_ptr(stream))
    if rc != FE_MF_OK:
        raise FeMfError(rc, "fe_mf_halo_add failed")
    return dst


def axpby(Z, W, beta: float, gamma: float, stream=None):
    """Z <- beta Z + gamma W on the device (fe_mf_axpby)."""
    import torch
    assert isinstance(Z, torch.Tensor) and Z.is_cuda and Z.dtype == torch.float64 and Z.is_contiguous()
    assert isinstance(W, torch.Tensor) and W.is_cuda and W.dtype == torch.float64 and W.is_contiguous()
    assert Z.numel() == W.numel()
    rc = lib().fe_mf_axpby(Z.data_ptr(), W.data_ptr(), float(beta), float(gamma), Z.numel(), _stream_ptr(stream))
    if rc != FE_MF_OK:
        raise FeMfError(rc, "fe_mf_axpby failed")
    return Z


def halo_pack_f32(dst, src, stream=None):
    """dst (float32) <- src (float64), round to nearest (fe_mf_halo_pack_f32): the sending side of the FP32 payload."""
    import torch
    assert isinstance(dst, torch.Tensor) and dst.is_cuda and dst.dtype == torch.float32 and dst.is_contiguous()
    assert isinstance(src, torch.Tensor) and src.is_cuda and src.dtype == torch.float64 and src.is_contiguous()
    assert dst.numel() == src.numel()
    rc = lib().fe_mf_halo_pack_f32(dst.data_ptr(), src.data_ptr(), dst.numel(), _stream_ptr(stream))
    if rc != FE_MF_OK:
        raise FeMfError(rc, "fe_mf_halo_pack_f32 failed")
    return dst


def halo_unpack_f32(dst, src, add: bool, stream=None):
    """dst (float64) <- src (float32), or dst += src (fe_mf_halo_unpack_f32): the receiving side of the FP32 payload."""
    import torch
    assert isinstance(dst, torch.Tensor) and dst.is_cuda and dst.dtype == torch.float64 and dst.is_contiguous()
    assert isinstance(src, torch.Tensor) and src.is_cuda and src.dtype == torch.float32 and src.is_contiguous()
    assert dst.numel() == src.numel()
    rc = lib().fe_mf_halo_unpack_f32(dst.data_ptr(), src.data_ptr(), dst.numel(), 1 if add else 0, _stream_ptr(stream))
    if rc != FE_MF_OK:
        raise FeMfError(rc, "fe_mf_halo_unpack_f32 failed")
    return dst


def probe_peaks(device: int = 0):
    """(FP64 FMA TFLOP/s, FP64 copy GB/s) measured live on `device`."""
    a, b = C.c_double(), C.c_double()
    rc = lib().fe_probe_peaks(C.byref(a), C.byref(b), int(device))
    if rc != FE_MF_OK:
        raise FeMfError(rc, "fe_probe_peaks failed")
    return a.value, b.value
