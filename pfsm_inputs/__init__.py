"""Seeded synthetic inputs for the PFSM path (recipe restated in DESIGN.md).

Draws numbers only -- none of the method's arithmetic lives here.  Shared by the oracle's
tests, the CUDA parity tests and bench.py, so that all of them see byte-identical matrices.

The paper's real matrices (RMG Kohn-Sham subspace Hamiltonians)
are not available; `config(k)` builds the synthetic stand-ins BASELINE.json:configs names:
A = diag(d) + E with E_ij = amp * N(0,1) * exp(-|i-j|/width), d shaped like the workload's
spectrum, alpha = 0.5 / max|d|^2.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pfsm_gen.c")
_LIB = os.path.join(_HERE, "libpfsm_gen.so")
_lib = None

SEED_BASE = 150207806
STREAM_D, STREAM_E, STREAM_S, STREAM_TEST = 0, 1, 2, 3


def build(force: bool = False) -> str:
    """Compile libpfsm_gen.so next to its source (gcc, seconds)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        u64, i64, dbl, p = ctypes.c_uint64, ctypes.c_int64, ctypes.c_double, ctypes.c_void_p
        lib.pfsm_gen_uniform.argtypes = [u64, u64, u64, i64, p]
        lib.pfsm_gen_normal.argtypes = [u64, u64, u64, i64, p]
        lib.pfsm_gen_banded_symmetric.argtypes = [i64, p, dbl, dbl, u64, u64, p]
        for f in (lib.pfsm_gen_uniform, lib.pfsm_gen_normal, lib.pfsm_gen_banded_symmetric):
            f.restype = None
        _lib = lib
    return _lib


def uniform(seed: int, stream: int, idx0: int, n: int) -> np.ndarray:
    out = np.empty(n, dtype=np.float64)
    _load().pfsm_gen_uniform(seed, stream, idx0, n, out.ctypes.data)
    return out


def normal(seed: int, stream: int, idx0: int, n: int) -> np.ndarray:
    out = np.empty(n, dtype=np.float64)
    _load().pfsm_gen_normal(seed, stream, idx0, n, out.ctypes.data)
    return out


def banded_symmetric(N: int, diag, amp: float, width: float, seed: int, stream: int,
                     out: np.ndarray | None = None) -> np.ndarray:
    """diag(diag) + amp * N(0,1) * exp(-|i-j|/width), exactly symmetric, shape (N, N)."""
    if out is None:
        out = np.empty((N, N), dtype=np.float64)
    assert out.shape == (N, N) and out.dtype == np.float64 and out.flags.c_contiguous
    dptr = None
    if diag is not None:
        diag = np.ascontiguousarray(diag, dtype=np.float64)
        assert diag.shape == (N,)
        dptr = diag.ctypes.data
    _load().pfsm_gen_banded_symmetric(N, dptr, amp, width, seed, stream, out.ctypes.data)
    return out


@dataclass
class Config:
    """One BASELINE.json config: shapes and PFSM parameters (no matrix yet)."""
    index: int
    name: str
    N: int
    P: int
    window: int
    iters: int
    amp: float
    width: float
    seed: int = field(init=False)

    def __post_init__(self):
        self.seed = SEED_BASE + self.index

    @property
    def m(self) -> int:
        return self.N // self.P

    @property
    def M(self) -> int:
        return min(self.N, self.m + 2 * self.window)


CONFIGS = [
    Config(0, "toy near-diagonal", 256, 4, 16, 3, 1e-3, 16.0),
    Config(1, "insulator (512-atom diamond shape)", 2048, 16, 32, 3, 1e-3, 32.0),
    Config(2, "molecular cluster (13xC60 shape)", 3072, 24, 48, 4, 5e-4, 64.0),
    Config(3, "many unoccupied states (Si216+vacancy shape)", 9072, 72, 64, 3, 1e-3, 64.0),
    Config(4, "metal, dense spectrum (Al4000 shape)", 8192, 64, 64, 5, 2e-3, 128.0),
]

# Beyond BASELINE.json: the size of the paper's Table I workload (256-atom copper cell with 256
# unoccupied orbitals, N = 1664) with the submatrix width the paper recommends, gamma = M / N = 0.25
# (PAPER.md:100-108): m = 128, window 144, M = 416.
EXTRA_CONFIGS = [
    Config(5, "transition metal with unoccupied states (Cu256 shape, Table I), gamma = 0.25", 1664, 13, 144, 3, 2e-3, 64.0),
    # config 4's workload (Al4000 shape, Table III) at the paper's recommended width gamma = M / N = 0.25
    # ("M <= 3000"): m = 512, window 768, M = 2048 -- the wide-window route of step 2
    Config(6, "metal, dense spectrum (Al4000 shape), gamma = 0.25", 8192, 16, 768, 3, 2e-3, 128.0),
]


def config(k: int) -> Config:
    """BASELINE.json config k (0-4) or an extra one (5, 6)."""
    return CONFIGS[k] if k < len(CONFIGS) else EXTRA_CONFIGS[k - len(CONFIGS)]


def spectrum(k: int) -> np.ndarray:
    """The intended eigenvalues d (sorted ascending) of config k -- SURVEY.md §8(d) table."""
    c = config(k)
    s, N = c.seed, c.N
    if k == 0:
        d = -1.0 + 2.0 * uniform(s, STREAM_D, 0, N)
    elif k == 1:
        occ = -0.8 + 1.1 * uniform(s, STREAM_D, 0, 1024)
        unocc = 0.5 + 1.5 * uniform(s, STREAM_D, 1024, 1024)
        d = np.concatenate([occ, unocc])
    elif k == 2:
        ncent = 237  # 236 * 13 + 4 = 3072
        centres = -1.0 + 2.5 * uniform(s, STREAM_D, 0, ncent)
        members = normal(s, STREAM_D, 1 << 20, ncent * 13).reshape(ncent, 13)
        d = (centres[:, None] + 1e-3 * members).reshape(-1)[:N]
    elif k == 3:
        occ = -0.6 + 0.8 * uniform(s, STREAM_D, 0, 432)
        u = uniform(s, STREAM_D, 432, 8640)
        unocc = (0.125 + 7.875 * u) ** (2.0 / 3.0)  # density ~ sqrt(E) on [0.25, 4]
        d = np.concatenate([occ, unocc])
    elif k == 4 or k == 6:
        u = uniform(s, STREAM_D, 0, N)
        d = -1.0 + 4.0 * u ** (2.0 / 3.0)  # density ~ sqrt(E + 1) on [-1, 3]
    elif k == 5:
        dband = -0.40 + 0.30 * uniform(s, STREAM_D, 0, 1280)       # narrow, dense d band: 5 states per atom
        u = uniform(s, STREAM_D, 1280, 384)
        spband = -0.80 + 2.0 * u ** (2.0 / 3.0)                     # free-electron-like s/p band, density ~ sqrt(E)
        d = np.concatenate([dband, spband])
    else:
        raise IndexError(k)
    d = np.sort(d)
    assert d.shape == (N,)
    return d


@dataclass
class Problem:
    cfg: Config
    d: np.ndarray          # intended spectrum, sorted
    A: np.ndarray          # (N, N) float64, exactly symmetric
    alpha: float           # 0.5 / max|d|^2  (reading R4)
    S: np.ndarray | None = None  # overlap matrix for the generalized variant (config 4g)

    @property
    def normF(self) -> float:
        return float(np.sqrt(np.sum(self.A * self.A)))


def alpha_rule(d: np.ndarray) -> float:
    return 0.5 / float(np.max(np.abs(d))) ** 2


def problem(k: int, generalized: bool = False, seed_offset: int = 0) -> Problem:
    """Matrix + parameters of config k.  seed_offset draws an independent matrix of the same
    shape (used for multi-GPU replicas: rank r solves problem(k, seed_offset=r))."""
    c = config(k)
    d = spectrum(k)
    seed = c.seed + 1000 * seed_offset
    A = banded_symmetric(c.N, d, c.amp, c.width, seed, STREAM_E)
    S = None
    if generalized:
        S = banded_symmetric(c.N, np.ones(c.N), 1e-4, 128.0, seed, STREAM_S)
    return Problem(c, d, A, alpha_rule(d), S)


def small_problem(N: int, amp: float, width: float, seed: int, lo: float = -1.0, hi: float = 1.0) -> Problem:
    """Config-0-shaped problem of any size (parity cases with ragged tiles)."""
    d = np.sort(lo + (hi - lo) * uniform(seed, STREAM_D, 0, N))
    A = banded_symmetric(N, d, amp, width, seed, STREAM_E)
    cfg = Config(-1, f"small N={N}", N, 1, 0, 0, amp, width)
    cfg.seed = seed
    return Problem(cfg, d, A, alpha_rule(d))


def householder_orthogonal(N: int, nreflect: int, seed: int) -> np.ndarray:
    """Q = H_1 H_2 ... H_k, H = I - 2 v v^T / (v^T v), v drawn from stream 3 (pin P4/P5 inputs)."""
    Q = np.eye(N)
    for r in range(nreflect):
        v = normal(seed, STREAM_TEST, r * N, N)
        v /= np.linalg.norm(v)
        Q = Q - 2.0 * np.outer(Q @ v, v)
    return Q
