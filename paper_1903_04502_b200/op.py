"""Thin Python binding of include/purify_op.h (ctypes).  Argument marshalling only: every step of
the path runs in the CUDA library (csrc/).  PyTorch provides device memory and streams.

There is NO CPU fallback: if libpurify_op.so is missing or there is no CUDA device, calls raise.
This module never imports oracle/.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpurify_op.so")

C64, C128 = 0, 1
ANALYTIC, TABLE = 0, 1
STAGES = ("pad", "fft", "degrid", "grid", "ifft", "crop", "permute", "zero")

# every symbol include/purify_op.h declares (checked by tests/test_abi.py)
SYMBOLS = (
    "purify_op_create", "purify_op_create_host", "purify_op_destroy", "purify_op_info",
    "purify_op_permutation", "purify_degrid", "purify_grid", "purify_normal",
    "purify_degrid_native", "purify_grid_native", "purify_permute_to_native",
    "purify_permute_from_native", "purify_degrid_host", "purify_grid_host", "purify_normal_host",
    "purify_stage_fourier_grid", "purify_stage_gridded", "purify_stage_times_ms",
    "purify_last_launch_count", "purify_strerror", "purify_last_error", "purify_version", "purify_op_norm",
    "purify_admm_fidelity_step", "purify_op_set_time_stages", "purify_ubench_fma", "purify_grid_dist", "purify_normal_dist",
)


class PurifyOpts(C.Structure):
    _fields_ = [("kernel_mode", C.c_int), ("table_samples_per_unit", C.c_int), ("chunk", C.c_int),
                ("time_stages", C.c_int), ("admm_unfused", C.c_int), ("force_tile_sorted", C.c_int),
                ("reserved", C.c_int * 2)]


class PurifyInfo(C.Structure):
    _fields_ = [("n", C.c_int), ("K", C.c_int), ("J", C.c_int), ("dtype", C.c_int), ("kernel_mode", C.c_int),
                ("table_samples_per_unit", C.c_int), ("M", C.c_longlong), ("tile", C.c_int), ("n_tiles", C.c_int),
                ("n_tiles_nonempty", C.c_int), ("n_items", C.c_int), ("poly_degree", C.c_int),
                ("poly_max_abs_err", C.c_double), ("device_bytes", C.c_longlong), ("max_tile_count", C.c_longlong),
                ("M_native", C.c_longlong), ("n_batches", C.c_longlong), ("layout", C.c_int), ("tile_h", C.c_int)]


ALLREDUCE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_longlong, C.c_int, C.c_void_p)


class PurifyError(RuntimeError):
    def __init__(self, status: int, what: str, detail: str):
        super().__init__(f"{what}: status {status} ({detail})")
        self.status = status


_lib = None


def load_library():
    """dlopen the C-ABI library and declare its signatures.  Fails loudly if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(
            f"{LIB_PATH} not found: build it with `python -m paper_1903_04502_b200.build` "
            "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, ip, ll = C.c_void_p, C.c_int, C.c_longlong
    L.purify_op_create.argtypes = [C.POINTER(vp), ip, ip, ip, ll, vp, vp, ip, C.POINTER(PurifyOpts), vp]
    L.purify_op_create_host.argtypes = L.purify_op_create.argtypes
    L.purify_op_destroy.argtypes = [vp]
    L.purify_op_info.argtypes = [vp, C.POINTER(PurifyInfo)]
    L.purify_op_permutation.argtypes = [vp, C.POINTER(vp)]
    for name in ("purify_degrid", "purify_grid", "purify_normal", "purify_degrid_native", "purify_grid_native",
                 "purify_permute_to_native", "purify_permute_from_native", "purify_degrid_host",
                 "purify_grid_host", "purify_normal_host", "purify_stage_fourier_grid", "purify_stage_gridded"):
        getattr(L, name).argtypes = [vp, vp, vp, vp]
        getattr(L, name).restype = ip
    L.purify_op_norm.argtypes = [vp, vp, ip, C.c_double, C.POINTER(C.c_double), C.POINTER(ip), vp]
    L.purify_op_norm.restype = ip
    L.purify_admm_fidelity_step.argtypes = [vp, vp, vp, vp, C.c_double, C.c_double, vp, C.POINTER(C.c_double), vp]
    L.purify_admm_fidelity_step.restype = ip
    for name in ("purify_grid_dist", "purify_normal_dist"):
        getattr(L, name).argtypes = [vp, vp, vp, ip, ALLREDUCE_FN, vp, vp]
        getattr(L, name).restype = ip
    L.purify_ubench_fma.argtypes = [ip, ip, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    L.purify_ubench_fma.restype = ip
    L.purify_stage_times_ms.argtypes = [vp, C.POINTER(C.c_float)]
    L.purify_op_set_time_stages.argtypes = [vp, ip]
    L.purify_op_set_time_stages.restype = ip
    L.purify_last_launch_count.argtypes = [vp]
    L.purify_strerror.argtypes = [ip]
    L.purify_strerror.restype = C.c_char_p
    L.purify_last_error.restype = C.c_char_p
    L.purify_version.restype = ip
    _lib = L
    return L


def _check(status: int, what: str):
    if status != 0:
        L = load_library()
        raise PurifyError(status, what, f"{L.purify_strerror(status).decode()}: {L.purify_last_error().decode()}")


def _stream() -> C.c_void_p:
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


_CDT = {C64: torch.complex64, C128: torch.complex128}
_RDT = {C64: torch.float32, C128: torch.float64}


class PurifyOp:
    """Handle of one measurement operator (purify_op_create ... purify_op_destroy)."""

    def __init__(self, n: int, J: int, uv: torch.Tensor, w: torch.Tensor | None = None, dtype: int = C64,
                 oversample: int = 2, kernel_mode: int = ANALYTIC, table_samples_per_unit: int = 0,
                 chunk: int = 0, time_stages: bool = False, admm_unfused: bool = False, tile_sorted: bool = False):
        self._L = load_library()
        self._h = C.c_void_p()
        self.n, self.K, self.J, self.dtype = int(n), 2 * int(n), int(J), int(dtype)
        opts = PurifyOpts(int(kernel_mode), int(table_samples_per_unit), int(chunk), int(bool(time_stages)),
                          int(bool(admm_unfused)), int(bool(tile_sorted)))
        M = 0 if uv is None else int(uv.shape[0])
        self.M = M
        rdt = _RDT.get(self.dtype, torch.float32)
        if uv is not None:
            if uv.dtype != rdt or uv.dim() != 2 or uv.shape[1] != 2 or not uv.is_contiguous():
                raise ValueError(f"uv must be a contiguous [M,2] {rdt} tensor")
        if w is not None:
            if w.dtype != rdt or w.shape != (M,) or not w.is_contiguous():
                raise ValueError(f"w must be a contiguous [M] {rdt} tensor")
        on_host = uv is not None and not uv.is_cuda
        if w is not None and uv is not None and w.is_cuda != uv.is_cuda:
            raise ValueError("uv and w must live on the same side (both host or both device)")
        fn = self._L.purify_op_create_host if on_host else self._L.purify_op_create
        st = fn(C.byref(self._h), int(n), int(oversample), int(J), M,
                C.c_void_p(uv.data_ptr()) if uv is not None and M > 0 else None,
                C.c_void_p(w.data_ptr()) if w is not None and M > 0 else None,
                int(dtype), C.byref(opts), _stream())
        _check(st, "purify_op_create")
        self.M_native = int(self.info()["M_native"])      # length of native-order vectors (>= M)

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._L.purify_op_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # -- facts
    def info(self) -> dict:
        inf = PurifyInfo()
        _check(self._L.purify_op_info(self._h, C.byref(inf)), "purify_op_info")
        return {k: getattr(inf, k) for k, _ in PurifyInfo._fields_}

    def permutation(self) -> torch.Tensor:
        """native -> caller index, as an int64 tensor of M_native entries on the device (copy);
        -1 marks a padding entry of the batched layout."""
        p = C.c_void_p()
        _check(self._L.purify_op_permutation(self._h, C.byref(p)), "purify_op_permutation")
        if self.M_native == 0:
            return torch.empty(0, dtype=torch.int64, device="cuda")
        view = torch.as_tensor(_DeviceArray(p.value, self.M_native, "<i4"), device="cuda")   # zero-copy view
        out = view.to(torch.int64) & 0xFFFFFFFF
        out[out == 0xFFFFFFFF] = -1
        return out

    def stage_times_ms(self) -> dict:
        arr = (C.c_float * 8)()
        _check(self._L.purify_stage_times_ms(self._h, arr), "purify_stage_times_ms")
        return {STAGES[i]: float(arr[i]) for i in range(8)}

    def set_time_stages(self, enable: bool):
        _check(self._L.purify_op_set_time_stages(self._h, int(bool(enable))), "purify_op_set_time_stages")

    def last_launch_count(self) -> int:
        return int(self._L.purify_last_launch_count(self._h))

    # -- helpers
    def _x(self, x, name="x"):
        if x.dtype != _CDT[self.dtype] or x.numel() != self.n * self.n or not x.is_contiguous():
            raise ValueError(f"{name} must be a contiguous {self.n}x{self.n} {_CDT[self.dtype]} tensor")
        return C.c_void_p(x.data_ptr())

    def _y(self, y, name="y", native=False):
        m = self.M_native if native else self.M
        if y.dtype != _CDT[self.dtype] or y.numel() != m or not y.is_contiguous():
            raise ValueError(f"{name} must be a contiguous [{m}] {_CDT[self.dtype]} tensor")
        return C.c_void_p(y.data_ptr()) if m > 0 else None

    def _new_x(self, device="cuda"):
        return torch.empty((self.n, self.n), dtype=_CDT[self.dtype], device=device)

    def _new_y(self, device="cuda", native=False):
        return torch.empty(self.M_native if native else self.M, dtype=_CDT[self.dtype], device=device)

    @staticmethod
    def _dev(*ts):
        for t in ts:
            if not t.is_cuda:
                raise ValueError("device entry point called with a host tensor (use the *_host methods)")

    # -- Phi, Phi^dagger, Phi^dagger Phi (device buffers)
    def degrid(self, x, y=None, native=False):
        y = self._new_y(native=native) if y is None else y
        self._dev(x, y)
        fn = self._L.purify_degrid_native if native else self._L.purify_degrid
        _check(fn(self._h, self._x(x), self._y(y, native=native), _stream()), "purify_degrid")
        return y

    def grid(self, y, x=None, native=False):
        x = self._new_x() if x is None else x
        self._dev(x, y)
        fn = self._L.purify_grid_native if native else self._L.purify_grid
        _check(fn(self._h, self._y(y, native=native), self._x(x), _stream()), "purify_grid")
        return x

    def normal(self, x, out=None):
        out = self._new_x() if out is None else out
        self._dev(x, out)
        _check(self._L.purify_normal(self._h, self._x(x), self._x(out, "out"), _stream()), "purify_normal")
        return out

    # -- f3: distributed-image operator; `allreduce(band: torch.Tensor)` sums a real view of one image band over the ranks
    def _dist_cb(self, out, allreduce):
        """ctypes callback that turns (pointer, count, stream) into a tensor view of `out` on that stream."""
        if allreduce is None:
            return C.cast(None, ALLREDUCE_FN)
        flat = torch.view_as_real(out).reshape(-1)
        base, item = flat.data_ptr(), flat.element_size()

        def cb(_user, ptr, count, _is_double, stream):
            try:
                off = (int(ptr) - base) // item
                with torch.cuda.stream(torch.cuda.ExternalStream(int(stream or 0))):
                    allreduce(flat[off:off + int(count)])
                return 0
            except Exception:           # never let an exception cross the C boundary
                import traceback
                traceback.print_exc()
                return 1
        return ALLREDUCE_FN(cb)

    def grid_dist(self, y_native, x=None, allreduce=None, bands: int = 4):
        x = self._new_x() if x is None else x
        self._dev(x, y_native)
        cb = self._dist_cb(x, allreduce)
        _check(self._L.purify_grid_dist(self._h, self._y(y_native, "y_native", True), self._x(x), int(bands), cb, None, _stream()),
               "purify_grid_dist")
        return x

    def normal_dist(self, x, out=None, allreduce=None, bands: int = 4):
        out = self._new_x() if out is None else out
        self._dev(x, out)
        cb = self._dist_cb(out, allreduce)
        _check(self._L.purify_normal_dist(self._h, self._x(x), self._x(out, "out"), int(bands), cb, None, _stream()),
               "purify_normal_dist")
        return out

    def permute_to_native(self, y, out=None):
        out = self._new_y(native=True) if out is None else out
        self._dev(y, out)
        _check(self._L.purify_permute_to_native(self._h, self._y(y), self._y(out, "out", True), _stream()), "permute_to_native")
        return out

    def permute_from_native(self, y, out=None):
        out = self._new_y() if out is None else out
        self._dev(y, out)
        _check(self._L.purify_permute_from_native(self._h, self._y(y, "y", True), self._y(out), _stream()), "permute_from_native")
        return out

    # -- host-buffer (end-to-end) entry points
    def degrid_host(self, x, y=None):
        y = self._new_y("cpu").pin_memory() if y is None else y
        _check(self._L.purify_degrid_host(self._h, self._x(x), self._y(y), _stream()), "purify_degrid_host")
        return y

    def grid_host(self, y, x=None):
        x = self._new_x("cpu").pin_memory() if x is None else x
        _check(self._L.purify_grid_host(self._h, self._y(y), self._x(x), _stream()), "purify_grid_host")
        return x

    def normal_host(self, x, out=None):
        out = self._new_x("cpu").pin_memory() if out is None else out
        _check(self._L.purify_normal_host(self._h, self._x(x), self._x(out, "out"), _stream()), "purify_normal_host")
        return out

    # -- f2: operator norm (largest eigenvalue of Phi^dagger Phi) by the power method
    def norm(self, x0=None, max_iter: int = 100, rel_tol: float = 1e-6):
        """Returns (lambda, iterations).  x0: n x n complex start vector on the device, or None for all ones."""
        lam, its = C.c_double(0.0), C.c_int(0)
        if x0 is not None:
            self._dev(x0)
        _check(self._L.purify_op_norm(self._h, self._x(x0, "x0") if x0 is not None else None, int(max_iter),
                                      float(rel_tol), C.byref(lam), C.byref(its), _stream()), "purify_op_norm")
        return float(lam.value), int(its.value)

    # -- f1: data-fidelity half of one ADMM iteration (Algorithm 1 lines 3-6), native-order y and s (s updated in place)
    def admm_fidelity_step(self, x, y_native, s_native, epsilon: float, varrho: float, g=None, want_norm: bool = True):
        """Returns (g, ||v + s_old - y||_2 or None) with g = Phi^dagger (v - r + s_new); s_native is updated in place."""
        g = self._new_x() if g is None else g
        self._dev(x, y_native, s_native, g)
        nrm = C.c_double(0.0)
        _check(self._L.purify_admm_fidelity_step(self._h, self._x(x), self._y(y_native, "y_native", True),
                                                 self._y(s_native, "s_native", True), float(epsilon), float(varrho),
                                                 self._x(g, "g"), C.byref(nrm) if want_norm else None, _stream()),
               "purify_admm_fidelity_step")
        return g, (float(nrm.value) if want_norm else None)

    # -- single stages in the mathematical layout (tests)
    def stage_fourier_grid(self, x):
        B = torch.empty((self.K, self.K), dtype=_CDT[self.dtype], device="cuda")
        _check(self._L.purify_stage_fourier_grid(self._h, self._x(x), C.c_void_p(B.data_ptr()), _stream()),
               "purify_stage_fourier_grid")
        return B

    def stage_gridded(self, y):
        B = torch.empty((self.K, self.K), dtype=_CDT[self.dtype], device="cuda")
        _check(self._L.purify_stage_gridded(self._h, self._y(y), C.c_void_p(B.data_ptr()), _stream()),
               "purify_stage_gridded")
        return B


UBENCH_FORMS = ("2 x FFMA, 3 registers", "FFMA2 broadcast scalar x pair + pair (degridding row pass)",
                "FFMA2 pair x pair + pair (weight combination)", "FFMA2 pair x pair + constant (Horner step)",
                "FFMA2 varying scalar x shared pair + pair (gridding)")


def ubench_fma(form: int, warps_per_sm: int = 16):
    """(SM cycles per warp instruction per SM sub-partition, SM clock in GHz) of one packed-fp32 instruction form."""
    L = load_library()
    cyc, ghz = C.c_double(0.0), C.c_double(0.0)
    _check(L.purify_ubench_fma(int(form), int(warps_per_sm), C.byref(cyc), C.byref(ghz)), "purify_ubench_fma")
    return float(cyc.value), float(ghz.value)


class _DeviceArray:
    """__cuda_array_interface__ wrapper of a library-owned device pointer."""

    def __init__(self, ptr: int, count: int, typestr: str):
        self.__cuda_array_interface__ = {"shape": (count,), "typestr": typestr, "data": (ptr, False), "version": 2}
