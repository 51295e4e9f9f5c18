"""pfsm_rayleigh_noalloc -- the one entry point that allocates nothing (static device scratch inside the library) --
against the existing step-5 path (pfsm_rayleigh through a handle), on two calls in a row.

Collected last on purpose (pytest -x: a failure here must not hide other tests).  Passes alone in a
fresh process and after the rest of the suite: it depends on no state but the library's own static array, which every
call overwrites before reading."""
import ctypes

import numpy as np
import pytest
import torch

import oracle
import pfsm_inputs as gen

pytestmark = pytest.mark.gpu

pfsm = pytest.importorskip("paper_1502_07806_b200")


def _existing_path(A, X):
    N = A.shape[0]
    h = pfsm.Handle(N, 1, 0, 0, 1.0)
    dl = torch.empty(N, dtype=torch.float64, device="cuda")
    h.rayleigh(torch.from_numpy(A).cuda(), torch.from_numpy(X).cuda(), dl)
    lam, res = dl.cpu().numpy(), h.residuals().cpu().numpy().copy()
    h.destroy()
    return lam, res


def _inputs(N, seed):
    p = gen.small_problem(N, 0.05, 10.0, seed=seed)
    X = gen.normal(seed, gen.STREAM_TEST, 0, N * N).reshape(N, N)
    X /= np.linalg.norm(X, axis=1, keepdims=True)
    return p.A, np.ascontiguousarray(X)


def test_no_alloc_entry_point_matches_existing_path_on_two_calls_in_a_row():
    # call 1 at the maximum size fills the whole static array; call 2, smaller and with other data, finds call 1's
    # contents there (the array is never cleared: every call overwrites what it reads) and must be just as right
    cases = [(1024, 41), (320, 42)]
    bufs = []
    for N, seed in cases:
        A, X = _inputs(N, seed)
        bufs.append((A, X, torch.from_numpy(A).cuda(), torch.from_numpy(X).cuda(),
                     torch.full((N,), float("nan"), dtype=torch.float64, device="cuda"),
                     torch.full((N,), float("nan"), dtype=torch.float64, device="cuda")))
    # warm-up call (first use loads the kernels, which may take device memory: not an allocation of the entry point's)
    pfsm.rayleigh_noalloc(bufs[1][2], bufs[1][3], bufs[1][4], bufs[1][5])
    torch.cuda.synchronize()
    bufs[1][4].fill_(float("nan"))
    bufs[1][5].fill_(float("nan"))
    free0 = torch.cuda.mem_get_info()[0]
    for A, X, dA, dX, dl, dr in bufs:                       # the two calls in a row, same stream
        pfsm.rayleigh_noalloc(dA, dX, dl, dr)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0            # no device memory was taken or given back
    for A, X, dA, dX, dl, dr in bufs:
        lam, res = dl.cpu().numpy(), dr.cpu().numpy()
        lam_ref, res_ref = _existing_path(A, X)
        assert np.abs(lam - lam_ref).max() < 1e-13          # (same kernels, same order: in fact the same bits)
        assert np.abs(res - res_ref).max() < 1e-13
        lam_o, res_o = oracle.step5(A, X)                   # and the oracle's definition, as the step-5 parity test does
        assert np.abs(lam - lam_o).max() < 1e-13
        assert np.abs(res - res_o).max() < 1e-13


def test_no_alloc_entry_point_rejects_sizes_beyond_its_static_scratch():
    lib = pfsm.load()
    buf = torch.zeros(16, dtype=torch.float64, device="cuda")
    ptr = ctypes.c_void_p(buf.data_ptr())
    for N in (1026, 2048, 255, 1, 0):                        # too large; odd (16-byte row pitch of the tensor maps); too small
        rc = lib.pfsm_rayleigh_noalloc(N, ptr, ptr, ptr, ptr, None)
        assert rc == pfsm.ERR_NOALLOC_SIZE
    assert "1024" in pfsm.strerror(pfsm.ERR_NOALLOC_SIZE)
    assert lib.pfsm_rayleigh_noalloc(64, None, ptr, ptr, ptr, None) == -2
    with pytest.raises(pfsm.PfsmError):
        N = 1026
        z = torch.zeros((N, N), dtype=torch.float64, device="cuda")
        v = torch.zeros(N, dtype=torch.float64, device="cuda")
        pfsm.rayleigh_noalloc(z, z, v, v)
