"""Thin Python binding of include/purify_wavelet.h (ctypes): the wavelet dictionary Psi / Psi^dagger (Dirac +
Daubechies 1-8) and one Dual Forward-Backward pass (Algorithm 1 lines 12-13).  Argument marshalling only: every step
runs in the CUDA library (csrc/wavelet.cu).  No CPU fallback; never imports oracle/."""
from __future__ import annotations

import ctypes as C

import torch

from .op import C64, C128, _CDT, _check, _stream, load_library

N_BASES = 9
SYMBOLS = ("purify_wavelet_create", "purify_wavelet_destroy", "purify_wavelet_filter", "purify_wavelet_adjoint",
           "purify_wavelet_forward", "purify_dualfb_step", "purify_project_positive")


def _lib():
    L = load_library()
    if not getattr(L, "_wavelet_declared", False):
        vp, ip = C.c_void_p, C.c_int
        L.purify_wavelet_create.argtypes = [C.POINTER(vp), ip, ip, ip, vp]
        L.purify_wavelet_destroy.argtypes = [vp]
        L.purify_wavelet_filter.argtypes = [vp, ip, C.POINTER(C.c_double)]
        L.purify_wavelet_adjoint.argtypes = [vp, vp, vp, vp]
        L.purify_wavelet_forward.argtypes = [vp, vp, vp, vp]
        L.purify_dualfb_step.argtypes = [vp, vp, vp, vp, vp, C.c_double, C.c_double, vp]
        L.purify_project_positive.argtypes = [vp, vp, vp, vp]
        for s in SYMBOLS:
            getattr(L, s).restype = ip
        L._wavelet_declared = True
    return L


class Wavelet:
    """Handle of the dictionary for n x n images (purify_wavelet_create ... purify_wavelet_destroy)."""

    def __init__(self, n: int, levels: int = 3, dtype: int = C64):
        self._L = _lib()
        self._h = C.c_void_p()
        self.n, self.levels, self.dtype = int(n), int(levels), int(dtype)
        _check(self._L.purify_wavelet_create(C.byref(self._h), self.n, self.levels, self.dtype, _stream()), "purify_wavelet_create")

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._L.purify_wavelet_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def filter(self, basis: int):
        buf = (C.c_double * 16)()
        n = self._L.purify_wavelet_filter(self._h, int(basis), buf)
        if n < 0:
            _check(n, "purify_wavelet_filter")
        return [float(buf[i]) for i in range(n)]

    def _img(self, t, name):
        if not t.is_cuda or t.dtype != _CDT[self.dtype] or t.numel() != self.n * self.n or not t.is_contiguous():
            raise ValueError(f"{name} must be a contiguous {self.n}x{self.n} {_CDT[self.dtype]} CUDA tensor")
        return C.c_void_p(t.data_ptr())

    def _coef(self, t, name):
        if not t.is_cuda or t.dtype != _CDT[self.dtype] or t.numel() != N_BASES * self.n * self.n or not t.is_contiguous():
            raise ValueError(f"{name} must be a contiguous [9,{self.n},{self.n}] {_CDT[self.dtype]} CUDA tensor")
        return C.c_void_p(t.data_ptr())

    def new_image(self):
        return torch.empty((self.n, self.n), dtype=_CDT[self.dtype], device="cuda")

    def new_coefficients(self):
        return torch.empty((N_BASES, self.n, self.n), dtype=_CDT[self.dtype], device="cuda")

    def adjoint(self, x, alpha=None):
        """alpha = Psi^dagger x"""
        alpha = self.new_coefficients() if alpha is None else alpha
        _check(self._L.purify_wavelet_adjoint(self._h, self._img(x, "x"), self._coef(alpha, "alpha"), _stream()), "purify_wavelet_adjoint")
        return alpha

    def forward(self, alpha, x=None):
        """x = Psi alpha"""
        x = self.new_image() if x is None else x
        _check(self._L.purify_wavelet_forward(self._h, self._coef(alpha, "alpha"), self._img(x, "x"), _stream()), "purify_wavelet_forward")
        return x

    def project_positive(self, z, out=None):
        out = self.new_image() if out is None else out
        _check(self._L.purify_project_positive(self._h, self._img(z, "z"), self._img(out, "out"), _stream()), "purify_project_positive")
        return out

    def dualfb_step(self, z, zbar_prev, d, gamma: float, eta: float, zbar_out=None):
        """One pass of Algorithm 1 lines 12-13; d is updated in place; returns zbar."""
        zbar_out = self.new_image() if zbar_out is None else zbar_out
        _check(self._L.purify_dualfb_step(self._h, self._img(z, "z"), self._img(zbar_prev, "zbar_prev"), self._coef(d, "d"),
                                          self._img(zbar_out, "zbar_out"), float(gamma), float(eta), _stream()), "purify_dualfb_step")
        return zbar_out
