"""paper_1502_07806_b200 -- thin Python binding over libpfsm.so (include/pfsm.h).

Argument marshalling only: every step of the PFSM solve (arXiv 1502.07806 section II)
runs in the CUDA kernels behind the C ABI.  PyTorch is used for device memory and streams, nothing else.
There is no CPU fallback: if the library cannot be built/loaded, or CUDA is unavailable, calls raise.

Layout: the C ABI is column-major with eigenvector i at V + i*N.  A C-contiguous torch tensor `Vr` of
shape (N, N) whose ROW i is eigenvector i is exactly that memory.  A is symmetric (layout immaterial).
"""
from __future__ import annotations

import ctypes
import os

from . import build as _build

_lib = None
CUDA_ERROR_BASE = 1000

EXPORTS = [
    "pfsm_create", "pfsm_solve", "pfsm_solve_host", "pfsm_solve_partial", "pfsm_orthonormalize", "pfsm_rayleigh", "pfsm_solve_generalized",
    "pfsm_generalized_reduce", "pfsm_solve_warm", "pfsm_standard_form_eq14",
    "pfsm_set_shard", "pfsm_shard_phase", "pfsm_shard_buffer", "pfsm_destroy", "pfsm_get_info", "pfsm_check_validity",
    "pfsm_get_step2_sweeps", "pfsm_get_residuals", "pfsm_get_shifts", "pfsm_set_alpha", "pfsm_set_cholqr_passes", "pfsm_set_option", "pfsm_rayleigh_noalloc", "pfsm_ipc_export", "pfsm_ipc_open", "pfsm_ipc_close",
    "pfsm_set_shard_peers", "pfsm_workspace_bytes",
    "pfsm_launches_per_solve", "pfsm_enable_step_timing", "pfsm_get_step_ms", "pfsm_probe_fp64_peak",
    "pfsm_strerror",
]


class PfsmError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where} failed with code {code}: {strerror(code)}")


def lib_path() -> str:
    return _build.LIB


def load(build_if_missing: bool = True):
    """dlopen libpfsm.so and declare the prototypes of include/pfsm.h.  Raises if it cannot be loaded."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing and _build.stale():
        _build.build()
    if not os.path.exists(_build.LIB):
        raise RuntimeError(f"{_build.LIB} is missing: build it with `python -m paper_1502_07806_b200.build`")
    lib = ctypes.CDLL(_build.LIB)
    i32, i64, dbl, p = ctypes.c_int32, ctypes.c_int64, ctypes.c_double, ctypes.c_void_p
    lib.pfsm_create.argtypes = [ctypes.POINTER(p), i64, i32, i32, i32, dbl]
    lib.pfsm_solve.argtypes = [p, p, p, p, p]
    lib.pfsm_solve_host.argtypes = [p, p, p, p, p]
    lib.pfsm_solve_partial.argtypes = [p, p, p, p, p, i32]
    lib.pfsm_orthonormalize.argtypes = [p, p, p]
    lib.pfsm_rayleigh.argtypes = [p, p, p, p, p]
    lib.pfsm_solve_generalized.argtypes = [p, p, p, p, p, p]
    lib.pfsm_generalized_reduce.argtypes = [p, p, p, p, p]
    lib.pfsm_solve_warm.argtypes = [p, p, p, p, p]
    lib.pfsm_standard_form_eq14.argtypes = [p, p, p, p, i32, i32, p]
    lib.pfsm_set_shard.argtypes = [p, i32, i32]
    lib.pfsm_shard_phase.argtypes = [p, i32, p, p, p, p]
    lib.pfsm_shard_buffer.argtypes = [p, i32, ctypes.POINTER(p)]
    lib.pfsm_destroy.argtypes = [p]
    lib.pfsm_get_info.argtypes = [p, p, ctypes.POINTER(i64)]
    lib.pfsm_get_step2_sweeps.argtypes = [p, p, ctypes.POINTER(i32)]
    lib.pfsm_check_validity.argtypes = [p, p, dbl, ctypes.POINTER(i32), ctypes.POINTER(dbl), ctypes.POINTER(i64)]
    lib.pfsm_get_residuals.argtypes = [p, ctypes.POINTER(p)]
    lib.pfsm_get_shifts.argtypes = [p, ctypes.POINTER(p)]
    lib.pfsm_set_alpha.argtypes = [p, dbl]
    lib.pfsm_set_cholqr_passes.argtypes = [p, i32]
    lib.pfsm_set_option.argtypes = [p, ctypes.c_char_p, i64]
    lib.pfsm_rayleigh_noalloc.argtypes = [i64, p, p, p, p, p]
    lib.pfsm_ipc_export.argtypes = [p, p, ctypes.POINTER(i64)]
    lib.pfsm_ipc_open.argtypes = [p, i64, ctypes.POINTER(p), ctypes.POINTER(p)]
    lib.pfsm_ipc_close.argtypes = [p]
    lib.pfsm_set_shard_peers.argtypes = [p, i32, ctypes.POINTER(p), i32]
    lib.pfsm_workspace_bytes.argtypes = [p]
    lib.pfsm_workspace_bytes.restype = ctypes.c_size_t
    lib.pfsm_launches_per_solve.argtypes = [p]
    lib.pfsm_launches_per_solve.restype = i64
    lib.pfsm_enable_step_timing.argtypes = [p, i32]
    lib.pfsm_get_step_ms.argtypes = [p, ctypes.POINTER(ctypes.c_float)]
    lib.pfsm_probe_fp64_peak.argtypes = [i32, p, ctypes.POINTER(dbl)]
    lib.pfsm_strerror.argtypes = [ctypes.c_int]
    lib.pfsm_strerror.restype = ctypes.c_char_p
    for name in EXPORTS:
        if name not in ("pfsm_workspace_bytes", "pfsm_launches_per_solve", "pfsm_strerror"):
            getattr(lib, name).restype = ctypes.c_int
    _lib = lib
    return lib


def strerror(code: int) -> str:
    return load().pfsm_strerror(code).decode()


def _check(code: int, where: str):
    if code != 0:
        raise PfsmError(code, where)


def _stream_ptr(stream) -> int:
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


def _dev_ptr(t, N, shape, name):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
            and tuple(t.shape) == shape):
        raise TypeError(f"{name}: need a contiguous CUDA float64 tensor of shape {shape}")
    return t.data_ptr()


def _host_ptr(t, shape, name):
    import torch
    if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
            and tuple(t.shape) == shape):
        raise TypeError(f"{name}: need a contiguous CPU float64 tensor of shape {shape}")
    return t.data_ptr()


class Handle:
    """Owns a pfsm_handle_t.  Mirrors the C ABI one to one; see include/pfsm.h for semantics."""

    def __init__(self, N: int, P: int, window: int, iters: int, alpha: float, options: dict | None = None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1502_07806_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        self._lib = load()
        self._h = ctypes.c_void_p()
        _check(self._lib.pfsm_create(ctypes.byref(self._h), N, P, window, iters, alpha), "pfsm_create")
        self.N, self.P, self.window, self.iters, self.alpha = N, P, window, iters, alpha
        for key, value in (options or {}).items():
            self.set_option(key, value)

    def solve(self, A, Vr, lam, stream=None):
        N = self.N
        _check(self._lib.pfsm_solve(self._h, _dev_ptr(A, N, (N, N), "A"), _dev_ptr(Vr, N, (N, N), "V"),
                                    _dev_ptr(lam, N, (N,), "lambda"), _stream_ptr(stream)), "pfsm_solve")

    def solve_partial(self, A, Vr, lam, last_step: int, stream=None):
        N = self.N
        lp = _dev_ptr(lam, N, (N,), "lambda") if lam is not None else None
        _check(self._lib.pfsm_solve_partial(self._h, _dev_ptr(A, N, (N, N), "A"), _dev_ptr(Vr, N, (N, N), "V"),
                                            lp, _stream_ptr(stream), last_step), "pfsm_solve_partial")

    def orthonormalize(self, Vr, stream=None):
        N = self.N
        _check(self._lib.pfsm_orthonormalize(self._h, _dev_ptr(Vr, N, (N, N), "V"), _stream_ptr(stream)),
               "pfsm_orthonormalize")

    def rayleigh(self, A, Vr, lam, stream=None):
        N = self.N
        _check(self._lib.pfsm_rayleigh(self._h, _dev_ptr(A, N, (N, N), "A"), _dev_ptr(Vr, N, (N, N), "V"),
                                       _dev_ptr(lam, N, (N,), "lambda"), _stream_ptr(stream)), "pfsm_rayleigh")

    def solve_generalized(self, A, S, Xr, lam, stream=None):
        N = self.N
        _check(self._lib.pfsm_solve_generalized(self._h, _dev_ptr(A, N, (N, N), "A"), _dev_ptr(S, N, (N, N), "S"),
                                                _dev_ptr(Xr, N, (N, N), "X"), _dev_ptr(lam, N, (N,), "lambda"),
                                                _stream_ptr(stream)), "pfsm_solve_generalized")

    def generalized_reduce(self, A, S, Ap, stream=None):
        N = self.N
        _check(self._lib.pfsm_generalized_reduce(self._h, _dev_ptr(A, N, (N, N), "A"), _dev_ptr(S, N, (N, N), "S"),
                                                 _dev_ptr(Ap, N, (N, N), "Ap"), _stream_ptr(stream)),
               "pfsm_generalized_reduce")

    def solve_warm(self, A, Vr, lam, stream=None):
        """SCF-sequence mode: Vr holds the previous step's orthonormal eigenvectors on input."""
        N = self.N
        _check(self._lib.pfsm_solve_warm(self._h, _dev_ptr(A, N, (N, N), "A"), _dev_ptr(Vr, N, (N, N), "V"),
                                         _dev_ptr(lam, N, (N,), "lambda"), _stream_ptr(stream)), "pfsm_solve_warm")

    def standard_form_eq14(self, A, B, Z, niter: int, symmetrize: bool = True, stream=None):
        N = self.N
        _check(self._lib.pfsm_standard_form_eq14(self._h, _dev_ptr(A, N, (N, N), "A"), _dev_ptr(B, N, (N, N), "B"),
                                                 _dev_ptr(Z, N, (N, N), "Z"), niter, int(symmetrize),
                                                 _stream_ptr(stream)), "pfsm_standard_form_eq14")

    def set_shard(self, rank: int, world: int):
        _check(self._lib.pfsm_set_shard(self._h, rank, world), "pfsm_set_shard")

    def shard_phase(self, phase: int, A, Vr, lam, stream=None):
        N = self.N
        ap = _dev_ptr(A, N, (N, N), "A") if A is not None else None
        lp = _dev_ptr(lam, N, (N,), "lambda") if lam is not None else None
        _check(self._lib.pfsm_shard_phase(self._h, phase, ap, _dev_ptr(Vr, N, (N, N), "V"), lp, _stream_ptr(stream)),
               "pfsm_shard_phase")

    def set_shard_peers(self, which: int, ptrs):
        arr = (ctypes.c_void_p * max(1, len(ptrs)))(*ptrs)
        _check(self._lib.pfsm_set_shard_peers(self._h, which, arr, len(ptrs)), "pfsm_set_shard_peers")

    def shard_buffer(self, which: int):
        """Zero-copy (N, N) tensor view of a handle-owned exchange buffer (0: G, 1: V^T R^-1)."""
        import torch
        ptr = ctypes.c_void_p()
        _check(self._lib.pfsm_shard_buffer(self._h, which, ctypes.byref(ptr)), "pfsm_shard_buffer")

        class _DevBuf:
            __cuda_array_interface__ = {"shape": (self.N, self.N), "typestr": "<f8", "data": (int(ptr.value), False),
                                        "version": 2}

        return torch.as_tensor(_DevBuf(), device="cuda")

    def residuals_view(self):
        """Zero-copy (N,) tensor view of the handle's residual buffer (for the sharded solve's all-gather)."""
        import torch
        ptr = ctypes.c_void_p()
        _check(self._lib.pfsm_get_residuals(self._h, ctypes.byref(ptr)), "pfsm_get_residuals")

        class _DevBuf:
            __cuda_array_interface__ = {"shape": (self.N,), "typestr": "<f8", "data": (int(ptr.value), False),
                                        "version": 2}

        return torch.as_tensor(_DevBuf(), device="cuda")

    def solve_host(self, A_host, Vr_host, lam_host, stream=None):
        N = self.N
        _check(self._lib.pfsm_solve_host(self._h, _host_ptr(A_host, (N, N), "A_host"),
                                         _host_ptr(Vr_host, (N, N), "V_host"), _host_ptr(lam_host, (N,), "lambda_host"),
                                         _stream_ptr(stream)), "pfsm_solve_host")

    def info(self, stream=None) -> int:
        v = ctypes.c_int64(-1)
        _check(self._lib.pfsm_get_info(self._h, _stream_ptr(stream), ctypes.byref(v)), "pfsm_get_info")
        return int(v.value)

    def check_validity(self, resid_tol: float, stream=None):
        """PAPER.md:98-100 guard.  Returns (use_standard_solver: bool, max_resid: float, info: int)."""
        verdict, mx, info = ctypes.c_int32(-1), ctypes.c_double(0.0), ctypes.c_int64(-1)
        _check(self._lib.pfsm_check_validity(self._h, _stream_ptr(stream), resid_tol, ctypes.byref(verdict),
                                             ctypes.byref(mx), ctypes.byref(info)), "pfsm_check_validity")
        return bool(verdict.value), float(mx.value), int(info.value)

    def _view(self, getter, name):
        import torch
        ptr = ctypes.c_void_p()
        _check(getter(self._h, ctypes.byref(ptr)), name)

        class _DevBuf:  # zero-copy view of the handle-owned device buffer, cloned into a tensor the caller owns
            __cuda_array_interface__ = {"shape": (self.N,), "typestr": "<f8", "data": (int(ptr.value), False),
                                        "version": 2}

        return torch.as_tensor(_DevBuf(), device="cuda").clone()

    def step2_sweeps(self, stream=None) -> int:
        v = ctypes.c_int32(0)
        _check(self._lib.pfsm_get_step2_sweeps(self._h, _stream_ptr(stream), ctypes.byref(v)), "pfsm_get_step2_sweeps")
        return int(v.value)

    def residuals(self):
        return self._view(self._lib.pfsm_get_residuals, "pfsm_get_residuals")

    def shifts(self):
        return self._view(self._lib.pfsm_get_shifts, "pfsm_get_shifts")

    def set_alpha(self, alpha: float):
        _check(self._lib.pfsm_set_alpha(self._h, alpha), "pfsm_set_alpha")
        self.alpha = alpha

    def set_option(self, key: str, value: int):
        _check(self._lib.pfsm_set_option(self._h, key.encode(), int(value)), f"pfsm_set_option({key!r}, {value})")

    def set_cholqr_passes(self, passes: int):
        _check(self._lib.pfsm_set_cholqr_passes(self._h, passes), "pfsm_set_cholqr_passes")

    def workspace_bytes(self) -> int:
        return int(self._lib.pfsm_workspace_bytes(self._h))

    def launches_per_solve(self) -> int:
        return int(self._lib.pfsm_launches_per_solve(self._h))

    def enable_step_timing(self, enable: bool = True):
        _check(self._lib.pfsm_enable_step_timing(self._h, int(enable)), "pfsm_enable_step_timing")

    def step_ms(self):
        arr = (ctypes.c_float * 4)()
        _check(self._lib.pfsm_get_step_ms(self._h, arr), "pfsm_get_step_ms")
        return [float(x) for x in arr]

    def destroy(self):
        if self._h:
            self._lib.pfsm_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


# Function-style aliases with the C names
def pfsm_create(N, P, window, iters, alpha) -> Handle:
    return Handle(N, P, window, iters, alpha)


def pfsm_solve(h: Handle, A, Vr, lam, stream=None):
    h.solve(A, Vr, lam, stream)


def pfsm_solve_host(h: Handle, A_host, Vr_host, lam_host, stream=None):
    h.solve_host(A_host, Vr_host, lam_host, stream)


def pfsm_destroy(h: Handle):
    h.destroy()


def probe_fp64_peak(kind: int = 0, stream=None) -> float:
    """TFLOP/s of a register-only FP64 loop on all SMs: kind 0 = DMMA (mma.sync m8n8k4 f64), 1 = DFMA."""
    v = ctypes.c_double(0.0)
    _check(load().pfsm_probe_fp64_peak(kind, _stream_ptr(stream), ctypes.byref(v)), "pfsm_probe_fp64_peak")
    return float(v.value)


ERR_NOALLOC_SIZE = 900


def rayleigh_noalloc(A, Vr, lam, resid, stream=None):
    """pfsm_rayleigh_noalloc: step 5 with no allocation anywhere (static device scratch inside the library; N even, <= 1024).
    A, Vr: (N, N) CUDA float64; lam, resid: (N,) CUDA float64 outputs.  Calls sharing a device must not overlap on the GPU."""
    N = A.shape[0]
    _check(load().pfsm_rayleigh_noalloc(N, _dev_ptr(A, N, (N, N), "A"), _dev_ptr(Vr, N, (N, N), "V"),
                                        _dev_ptr(lam, N, (N,), "lambda"), _dev_ptr(resid, N, (N,), "resid"),
                                        _stream_ptr(stream)), "pfsm_rayleigh_noalloc")


def ipc_export(t):
    """(64-byte handle, byte offset) of the CUDA allocation that holds tensor `t` -- plain Python values for all_gather_object."""
    buf = ctypes.create_string_buffer(64)
    off = ctypes.c_int64()
    _check(load().pfsm_ipc_export(t.data_ptr(), buf, ctypes.byref(off)), "pfsm_ipc_export")
    return bytes(buf.raw), int(off.value)


def ipc_open(handle: bytes, offset: int):
    """Maps another process's allocation; returns (base, ptr) as ints (pfsm_ipc_close takes base)."""
    base, ptr = ctypes.c_void_p(), ctypes.c_void_p()
    _check(load().pfsm_ipc_open(handle, offset, ctypes.byref(base), ctypes.byref(ptr)), "pfsm_ipc_open")
    return int(base.value), int(ptr.value)


def ipc_close(base: int):
    _check(load().pfsm_ipc_close(base), "pfsm_ipc_close")
