"""ctypes front-end of the CPU oracle (oracle/purify_oracle.cpp).

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this.  It shares nothing with the CUDA
path (paper_1903_04502_b200/csrc, paper_1903_04502_b200/op.py) and does not import it.

Everything is promoted to fp64 here: inputs stored as f32 / c64 are
converted exactly; `idx_prec` (32 for a C64 problem, 64 for C128) only selects the
precision in which the TABLE-mode lookup index is decided (purify_oracle.cpp KernelEval).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None
ANALYTIC, TABLE = 0, 1
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.oracle_num_threads.restype = C.c_int
        L.oracle_set_num_threads.argtypes = [C.c_int]
        L.oracle_i0.restype = C.c_double
        L.oracle_i0.argtypes = [C.c_double]
        L.oracle_kb.restype = C.c_double
        L.oracle_kb.argtypes = [C.c_double, C.c_int]
        L.oracle_kb_ghat.restype = C.c_double
        L.oracle_kb_ghat.argtypes = [C.c_double, C.c_int]
        L.oracle_correction.argtypes = [C.c_int, C.c_int, _dp]
        L.oracle_table_len.restype = C.c_long
        L.oracle_table_len.argtypes = [C.c_int, C.c_int]
        L.oracle_table.argtypes = [C.c_int, C.c_int, _dp]
        L.oracle_kernel_weight.restype = C.c_double
        L.oracle_kernel_weight.argtypes = [C.c_double, C.c_long, C.c_int, C.c_int, C.c_int, C.c_int]
        L.oracle_table_index.argtypes = [C.c_long, _dp, C.POINTER(C.c_long), C.c_int, C.c_int, C.POINTER(C.c_long)]
        L.oracle_fft2.argtypes = [_dp, C.c_int, C.c_int]
        L.oracle_dft2_direct.argtypes = [_dp, _dp, C.c_int, C.c_int]
        L.oracle_pad.argtypes = [C.c_int, C.c_int, _dp, _dp]
        L.oracle_crop.argtypes = [C.c_int, C.c_int, _dp, _dp]
        L.oracle_degrid_from_grid.argtypes = [C.c_int, C.c_int, C.c_long, _dp, _dp, _dp,
                                              C.c_int, C.c_int, C.c_int, _dp]
        L.oracle_grid_to_grid.argtypes = [C.c_int, C.c_int, C.c_long, _dp, _dp, _dp,
                                          C.c_int, C.c_int, C.c_int, _dp]
        L.oracle_degrid.argtypes = [C.c_int, C.c_int, C.c_long, _dp, _dp, _dp,
                                    C.c_int, C.c_int, C.c_int, _dp]
        L.oracle_grid.argtypes = [C.c_int, C.c_int, C.c_long, _dp, _dp, _dp,
                                  C.c_int, C.c_int, C.c_int, _dp]
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _c128(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def _mode(mode):
    if mode in ("analytic", ANALYTIC):
        return ANALYTIC
    if mode in ("table", TABLE):
        return TABLE
    raise ValueError(mode)


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_num_threads(t: int) -> None:
    lib().oracle_set_num_threads(int(t))


def i0(z: float) -> float:
    return float(lib().oracle_i0(float(z)))


def kb(d, J: int):
    """Kaiser-Bessel g(d), beta = 2.34 J (R1)."""
    L = lib()
    d = np.asarray(d, dtype=np.float64)
    return np.vectorize(lambda t: L.oracle_kb(float(t), int(J)), otypes=[np.float64])(d)


def kb_ghat(xi, J: int):
    """Continuous Fourier transform of g at frequency xi (cycles per cell) (R2)."""
    L = lib()
    xi = np.asarray(xi, dtype=np.float64)
    return np.vectorize(lambda t: L.oracle_kb_ghat(float(t), int(J)), otypes=[np.float64])(xi)


def correction(n: int, J: int) -> np.ndarray:
    s = np.empty(n, dtype=np.float64)
    lib().oracle_correction(int(n), int(J), _p(s))
    return s


def table(J: int, R: int) -> np.ndarray:
    L = lib()
    T = np.empty(L.oracle_table_len(int(J), int(R)), dtype=np.float64)
    L.oracle_table(int(J), int(R), _p(T))
    return T


def kernel_weight(u: float, c: int, J: int, mode="analytic", R: int = 4096, idx_prec: int = 64) -> float:
    return float(lib().oracle_kernel_weight(float(u), int(c), int(J), _mode(mode), int(R), int(idx_prec)))


def table_index(u, c, R: int = 4096, idx_prec: int = 64) -> np.ndarray:
    """R11: floor(|u - c| R + 1/2) for arrays of coordinates u and taps c, decided in fp32 (idx_prec 32) or fp64."""
    u = np.ascontiguousarray(u, dtype=np.float64)
    c = np.ascontiguousarray(c, dtype=np.int64)
    assert u.shape == c.shape and u.ndim == 1
    out = np.empty(len(u), dtype=np.int64)
    lp = C.POINTER(C.c_long)
    lib().oracle_table_index(len(u), _p(u), c.ctypes.data_as(lp), int(R), int(idx_prec), out.ctypes.data_as(lp))
    return out


def fft2(a: np.ndarray, sign: int = -1) -> np.ndarray:
    """Unnormalised 2-D DFT (sign -1 forward, +1 adjoint) of a K x K array (copy)."""
    out = _c128(a).copy()
    K = out.shape[0]
    assert out.shape == (K, K)
    lib().oracle_fft2(out.view(np.float64).ctypes.data_as(_dp), K, int(sign))
    return out


def dft2_direct(a: np.ndarray, sign: int = -1) -> np.ndarray:
    a = _c128(a)
    K = a.shape[0]
    out = np.empty_like(a)
    lib().oracle_dft2_direct(a.view(np.float64).ctypes.data_as(_dp),
                             out.view(np.float64).ctypes.data_as(_dp), K, int(sign))
    return out


def pad(x: np.ndarray, J: int) -> np.ndarray:
    x = _c128(x)
    n = x.shape[0]
    b = np.empty((2 * n, 2 * n), dtype=np.complex128)
    lib().oracle_pad(n, int(J), x.view(np.float64).ctypes.data_as(_dp), b.view(np.float64).ctypes.data_as(_dp))
    return b


def crop(b: np.ndarray, J: int) -> np.ndarray:
    b = _c128(b)
    n = b.shape[0] // 2
    x = np.empty((n, n), dtype=np.complex128)
    lib().oracle_crop(n, int(J), b.view(np.float64).ctypes.data_as(_dp), x.view(np.float64).ctypes.data_as(_dp))
    return x


def _uvw(uv, w):
    uv = np.ascontiguousarray(uv, dtype=np.float64)
    assert uv.ndim == 2 and uv.shape[1] == 2
    w = _f64(w)
    if w is not None:
        assert w.shape == (uv.shape[0],)
    return uv, w


def degrid_from_grid(B, uv, w, J, mode="analytic", R=4096, idx_prec=64) -> np.ndarray:
    """W G only: interpolate visibilities off a given K x K Fourier grid (O3 step 3)."""
    B = _c128(B)
    uv, w = _uvw(uv, w)
    y = np.empty(uv.shape[0], dtype=np.complex128)
    lib().oracle_degrid_from_grid(B.shape[0], int(J), uv.shape[0], B.view(np.float64).ctypes.data_as(_dp),
                                  _p(uv), _p(w), _mode(mode), int(R), int(idx_prec),
                                  y.view(np.float64).ctypes.data_as(_dp))
    return y


def grid_to_grid(y, uv, w, K, J, mode="analytic", R=4096, idx_prec=64) -> np.ndarray:
    """G^dagger W^dagger only: weighted gridding onto a K x K Fourier grid (O4 step 1)."""
    y = _c128(y)
    uv, w = _uvw(uv, w)
    Bp = np.empty((K, K), dtype=np.complex128)
    lib().oracle_grid_to_grid(int(K), int(J), uv.shape[0], y.view(np.float64).ctypes.data_as(_dp),
                              _p(uv), _p(w), _mode(mode), int(R), int(idx_prec),
                              Bp.view(np.float64).ctypes.data_as(_dp))
    return Bp


def degrid(x, uv, w, J, mode="analytic", R=4096, idx_prec=64) -> np.ndarray:
    """Phi x = W G F Z S x (Eq. 2)."""
    x = _c128(x)
    n = x.shape[0]
    assert x.shape == (n, n) and n % 2 == 0
    uv, w = _uvw(uv, w)
    y = np.empty(uv.shape[0], dtype=np.complex128)
    lib().oracle_degrid(n, int(J), uv.shape[0], x.view(np.float64).ctypes.data_as(_dp), _p(uv), _p(w),
                        _mode(mode), int(R), int(idx_prec), y.view(np.float64).ctypes.data_as(_dp))
    return y


def grid(y, uv, w, n, J, mode="analytic", R=4096, idx_prec=64) -> np.ndarray:
    """Phi^dagger y = S^dagger Z^dagger F^dagger G^dagger W^dagger y."""
    y = _c128(y)
    uv, w = _uvw(uv, w)
    x = np.empty((n, n), dtype=np.complex128)
    lib().oracle_grid(int(n), int(J), uv.shape[0], y.view(np.float64).ctypes.data_as(_dp), _p(uv), _p(w),
                      _mode(mode), int(R), int(idx_prec), x.view(np.float64).ctypes.data_as(_dp))
    return x


def power_method(x0, uv, w, n, J, max_iter=100, rel_tol=1e-6, mode="analytic", R=4096, idx_prec=64):
    """f2: largest eigenvalue of Phi^dagger Phi by the power method, step by step:
    x_1 = x0/||x0||; z_k = Phi^dagger Phi x_k; lambda_k = ||z_k||_2; x_{k+1} = z_k/lambda_k; stop after max_iter
    iterations or when |lambda_k - lambda_{k-1}| <= rel_tol lambda_k (k >= 2).  x0 None = all ones.
    Returns (lambda, iterations).  Pinned against numpy's dense eigen-solver on a tiny operator (tests)."""
    x = np.ones((n, n), dtype=np.complex128) if x0 is None else _c128(x0).copy()
    nrm = float(np.linalg.norm(x))
    assert nrm > 0.0
    lam = prev = 0.0
    it = 0
    for it in range(1, int(max_iter) + 1):
        x = x / nrm
        z = grid(degrid(x, uv, w, J, mode, R, idx_prec), uv, w, n, J, mode, R, idx_prec)
        prev, lam = lam, float(np.linalg.norm(z))
        x, nrm = z, lam
        if not lam > 0.0 or (it > 1 and abs(lam - prev) <= rel_tol * lam):
            break
    return lam, it


def admm_fidelity_step(x, y, s, uv, w, n, J, epsilon, varrho, mode="analytic", R=4096, idx_prec=64):
    """f1: Algorithm 1 lines 3-6 in the paper's order, caller-order vectors:
        v = Phi x                                    (line 3)
        r = P_B(v + s), ball of radius epsilon around y:  r = v + s if ||v + s - y|| <= epsilon,
                                                          else y + epsilon (v + s - y)/||v + s - y||   (line 4, Eq. 23)
        s_new = s + varrho (v - r)                   (line 5)
        g = Phi^dagger (v - r + s_new)               (line 6; the caller forms x~ = x - rho g)
    Returns (g, s_new, r, ||v + s - y||)."""
    y, s = _c128(y), _c128(s)
    v = degrid(x, uv, w, J, mode, R, idx_prec)
    d = v + s - y
    nrm = float(np.linalg.norm(d))
    r = v + s if nrm <= epsilon else y + d * (epsilon / nrm)
    s_new = s + varrho * (v - r)
    g = grid(v - r + s_new, uv, w, n, J, mode, R, idx_prec)
    return g, s_new, r, nrm
