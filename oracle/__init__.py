"""CPU oracle for the PFSM path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes binding over oracle/pfsm_oracle.cpp (plain C++17, FP64, OpenMP over independent
columns; see that file's header for the citation of every step and the list of pins).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package; it imports nothing from the CUDA package and shares no code with it.

Layout convention: the C code is column-major with eigenvector i at V + i*N.  On the numpy side
that is a C-contiguous array `Vr` of shape (N, N) whose ROW i is eigenvector i (Vr = V^T).  A is
symmetric, so its layout is immaterial.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pfsm_oracle.cpp")
_LIB = os.path.join(_HERE, "libpfsm_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", "-std=c++17", "-O2", "-march=x86-64-v3", "-fopenmp", "-fPIC", "-shared",
                               "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i64, dbl, p = ctypes.c_int64, ctypes.c_double, ctypes.c_void_p
        lib.oracle_partition.argtypes = [i64, i64, i64, p, p, p]
        lib.oracle_partition.restype = i64
        lib.oracle_jacobi_eig.argtypes = [i64, p, p, p]
        lib.oracle_jacobi_eig.restype = ctypes.c_int
        lib.oracle_step2.argtypes = [i64, i64, i64, p, p, p]
        lib.oracle_step2.restype = i64
        lib.oracle_step3.argtypes = [i64, i64, dbl, p, p, p, i64, i64]
        lib.oracle_step3.restype = None
        lib.oracle_step4_mgs.argtypes = [i64, i64, p]
        lib.oracle_step4_mgs.restype = i64
        lib.oracle_step5.argtypes = [i64, p, p, p, p, i64, i64]
        lib.oracle_step5.restype = None
        lib.oracle_pfsm.argtypes = [i64, i64, i64, i64, dbl, p, p, p, p, p]
        lib.oracle_pfsm.restype = i64
        lib.oracle_generalized_reduce.argtypes = [i64, p, p, p, p]
        lib.oracle_generalized_reduce.restype = i64
        lib.oracle_generalized_back.argtypes = [i64, p, p, p]
        lib.oracle_generalized_back.restype = None
        lib.oracle_eq14_iteration.argtypes = [i64, p, p, i64, p]
        lib.oracle_eq14_iteration.restype = None
        lib.oracle_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _f64(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        assert a.shape == shape, (a.shape, shape)
    return a


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def _partition_full(N: int, P: int, w: int):
    if P < 1:
        raise ValueError("invalid partition (P < 1)")
    g0 = np.zeros(P + 1, dtype=np.int64)
    lo, off = (np.zeros(P, dtype=np.int64) for _ in range(2))
    M = _load().oracle_partition(N, P, w, g0.ctypes.data, lo.ctypes.data, off.ctypes.data)
    if M < 0:
        raise ValueError("invalid partition (need 1 <= P <= N, w >= 0)")
    return int(M), g0, lo, off


def partition(N: int, P: int, w: int):
    """O1.  Returns (M, g0, lo, off) as int64 arrays of length P."""
    M, g0, lo, off = _partition_full(N, P, w)
    return M, g0[:P].copy(), lo, off


def slice_counts(N: int, P: int) -> np.ndarray:
    """Eigenpairs per slice, m_s = g0[s+1] - g0[s] (all N/P when P divides N; reading R14 otherwise)."""
    return np.diff(_partition_full(N, P, 0)[1])


def jacobi_eig(B):
    """O2/O6: full cyclic Jacobi eigendecomposition.  Returns (mu ascending, Y with eigenvectors as
    COLUMNS (numpy convention), sweeps)."""
    B = _f64(B).copy()
    n = B.shape[0]
    assert B.shape == (n, n)
    mu = np.empty(n)
    Yr = np.empty((n, n))  # C-order rows = column-major columns = eigenvectors
    sw = _load().oracle_jacobi_eig(n, B.ctypes.data, mu.ctypes.data, Yr.ctypes.data)
    return mu, Yr.T.copy(), int(sw)


def step2(A, P: int, w: int):
    """O2.  Returns (Vr, eps, info): Vr row i = zero-padded start vector x_i^0."""
    A = _f64(A)
    N = A.shape[0]
    Vr = np.empty((N, N))
    eps = np.empty(N)
    info = _load().oracle_step2(N, P, w, A.ctypes.data, Vr.ctypes.data, eps.ctypes.data)
    return Vr, eps, int(info)


def step3(A, Vr, eps, iters: int, alpha: float, c0: int = 0, c1: int | None = None):
    """O3 (Eq. 11) on rows [c0, c1) of Vr (eigenvectors c0..c1-1).  Returns a new array."""
    A = _f64(A)
    N = A.shape[0]
    Vr = _f64(Vr, (N, N)).copy()
    eps = _f64(eps, (N,))
    if c1 is None:
        c1 = N
    _load().oracle_step3(N, iters, alpha, A.ctypes.data, Vr.ctypes.data, eps.ctypes.data, c0, c1)
    return Vr


def step4_mgs(Vr, ncols: int | None = None):
    """O4: modified Gram-Schmidt over eigenvectors 0..ncols-1.  Returns (Vr, info)."""
    Vr = _f64(Vr).copy()
    ncols = Vr.shape[0] if ncols is None else ncols
    info = _load().oracle_step4_mgs(Vr.shape[1], ncols, Vr.ctypes.data)
    return Vr, int(info)


def step5(A, Vr, c0: int = 0, c1: int | None = None):
    """O5: Rayleigh quotients and residual norms of eigenvectors [c0, c1).  Returns (lambda, resid)
    (entries outside [c0, c1) are NaN)."""
    A = _f64(A)
    N = A.shape[0]
    Vr = _f64(Vr, (N, N))
    c1 = N if c1 is None else c1
    lam = np.full(N, np.nan)
    res = np.full(N, np.nan)
    _load().oracle_step5(N, A.ctypes.data, Vr.ctypes.data, lam.ctypes.data, res.ctypes.data, c0, c1)
    return lam, res


def pfsm(A, P: int, w: int, iters: int, alpha: float):
    """One PFSM solve, O1..O5.  Returns dict(Vr, lam, resid, eps, info)."""
    A = _f64(A)
    N = A.shape[0]
    Vr = np.zeros((N, N))
    lam, res, eps = np.zeros(N), np.zeros(N), np.zeros(N)
    info = _load().oracle_pfsm(N, P, w, iters, alpha, A.ctypes.data, Vr.ctypes.data, lam.ctypes.data,
                               res.ctypes.data, eps.ctypes.data)
    return dict(Vr=Vr, lam=lam, resid=res, eps=eps, info=int(info))


def generalized_reduce(A, S):
    """OG: S = L L^T, A' = L^-1 A L^-T (symmetrized).  Returns (L lower-triangular numpy matrix, A', info)."""
    A, S = _f64(A), _f64(S)
    N = A.shape[0]
    Lr = np.empty((N, N))  # column-major L == C-order L^T
    Ap = np.empty((N, N))
    info = _load().oracle_generalized_reduce(N, A.ctypes.data, S.ctypes.data, Lr.ctypes.data, Ap.ctypes.data)
    return Lr.T.copy(), Ap, int(info)


def generalized_back(L, Vr):
    """OG: X = L^-T V.  Vr rows = eigenvectors of A'; returns Xr rows = generalized eigenvectors."""
    L = _f64(L)
    N = L.shape[0]
    Lr = np.ascontiguousarray(L.T)  # column-major L
    Vr = _f64(Vr, (N, N))
    Xr = np.empty((N, N))
    _load().oracle_generalized_back(N, Lr.ctypes.data, Vr.ctypes.data, Xr.ctypes.data)
    return Xr


def pfsm_warm(A, Vr_prev, P: int, w: int, iters: int, alpha: float):
    """SCF-sequence mode: the previous step's orthonormal eigenvectors V_prev (rows of
    Vr_prev) make A' = V_prev^T A V_prev diagonally dominant; PFSM (O1..O5) runs on A', and the vectors are
    rotated back, V = V_prev U.  The two changes of basis are plain FP64 matrix products (library primitive)."""
    A = _f64(A)
    Vp = _f64(Vr_prev)
    Ap = Vp @ A @ Vp.T
    Ap = 0.5 * (Ap + Ap.T)
    r = pfsm(Ap, P, w, iters, alpha)
    r["Ur"] = r["Vr"]
    r["Vr"] = r["Ur"] @ Vp
    r["Ap"] = Ap
    return r


def eq14_iteration(A, B, niter: int, symmetrize: bool = False):
    """f2 (Eq. 14-15): Z_0 = A, Z <- Z - D^-1 (B Z - A), niter times.  Returns Z as a numpy
    matrix (Z[i, j]); symmetrize=True returns (Z + Z^T)/2, the matrix "used in Eq. (3)" (reading R19)."""
    A, B = _f64(A), _f64(B)
    N = A.shape[0]
    Zc = np.empty((N, N))  # column-major Z == C-order Z^T; A, B symmetric so their layout is immaterial
    _load().oracle_eq14_iteration(N, A.ctypes.data, B.ctypes.data, niter, Zc.ctypes.data)
    Z = Zc.T.copy()
    return 0.5 * (Z + Z.T) if symmetrize else Z
