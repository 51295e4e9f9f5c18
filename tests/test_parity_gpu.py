"""GPU parity: the CUDA path (through the C ABI of include/pfsm.h) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances are north_star's (reading R20):
    |lambda_gpu - lambda_oracle| <= 1e-10 ||A||_F        per index
    ||V^T V - I||_max            <= 1e-12 N              (GPU and oracle each)
    |r_gpu - r_oracle|           <= 1e-9 ||A||_F         per vector
Eigenvectors are compared up to their sign only where they are unique (reading R16)."""
import os

import numpy as np
import pytest
import torch

import oracle
import pfsm_inputs as gen

pytestmark = pytest.mark.gpu

pfsm = pytest.importorskip("paper_1502_07806_b200")


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


_ORACLE_MEMO = {}

# pfsm_set_option settings applied to every handle gpu_solve creates; tests select a kernel route with
# monkeypatch.setitem(OPTS, key, value) (include/pfsm.h lists the keys).  Empty = the product path.
OPTS = {}


def oracle_step2_memo(A, P, w):
    key = ("step2", A.shape[0], P, w, float(A.sum()), float(np.abs(A).sum()))
    if key not in _ORACLE_MEMO:
        _ORACLE_MEMO[key] = oracle.step2(A, P, w)
    return _ORACLE_MEMO[key]


def oracle_pfsm_memo(A, P, w, iters, alpha):
    """oracle.pfsm, computed once per input: tests parametrized over the step-2 route compare every route with the
    same oracle run (the oracle has one route)."""
    key = (A.shape[0], P, w, iters, float(alpha), float(A.sum()), float(np.abs(A).sum()))
    if key not in _ORACLE_MEMO:
        _ORACLE_MEMO[key] = oracle.pfsm(A, P, w, iters, alpha)
    return _ORACLE_MEMO[key]


def gpu_solve(A, P, w, iters, alpha, last_step=5):
    N = A.shape[0]
    h = pfsm.Handle(N, P, w, iters, alpha, options=OPTS)
    dA = dev(A)
    dV = torch.full((N, N), float("nan"), dtype=torch.float64, device="cuda")  # input content must be ignored (R13)
    dl = torch.full((N,), float("nan"), dtype=torch.float64, device="cuda")
    if last_step == 5:
        h.solve(dA, dV, dl)
    else:
        h.solve_partial(dA, dV, dl, last_step)
    info = h.info()
    out = dict(Vr=dV.cpu().numpy(), lam=dl.cpu().numpy(), resid=h.residuals().cpu().numpy(),
               eps=h.shifts().cpu().numpy(), info=info)
    h.destroy()
    return out


def align_signs(Vg, Vo):
    s = np.sign(np.einsum("ij,ij->i", Vg, Vo))
    s[s == 0] = 1.0
    return Vg * s[:, None]


def check_gates(p_A, g, o):
    N = p_A.shape[0]
    nF = float(np.linalg.norm(p_A))
    assert g["info"] == 0 and o["info"] == 0
    assert np.abs(g["lam"] - o["lam"]).max() <= 1e-10 * nF
    assert np.abs(g["Vr"] @ g["Vr"].T - np.eye(N)).max() <= 1e-12 * N
    assert np.abs(o["Vr"] @ o["Vr"].T - np.eye(N)).max() <= 1e-12 * N
    assert np.abs(g["resid"] - o["resid"]).max() <= 1e-9 * nF
    assert abs(g["lam"].sum() - np.trace(p_A)) <= 1e-11 * N * max(1.0, np.abs(np.diag(p_A)).max())  # P7


# shapes: several 128-tiles plus ragged tails; odd M; m not dividing the tile; slices straddling tiles
SMALL_CASES = [
    # N, P, w, iters, amp, width
    (256, 4, 16, 3, 1e-3, 16.0),     # BASELINE config 0 shape
    (304, 4, 10, 2, 2e-3, 12.0),     # ragged: 304 = 2*128 + 48, M = 96
    (270, 6, 4, 3, 1e-3, 8.0),       # m = 45, M = 53 (odd -> phantom column in the tournament)
    (400, 5, 24, 1, 1e-3, 16.0),     # M = 128
    (600, 3, 20, 2, 5e-4, 24.0),     # m = 200, M = 240, slices straddle tiles
    (130, 1, 0, 2, 1e-2, 8.0),       # P = 1: submatrix = A, PFSM exact (P3)
    (96, 4, 100, 2, 1e-2, 8.0),      # window >= N: every slice diagonalizes all of A
    (64, 8, 0, 4, 1e-3, 4.0),        # window 0: M = m
    (2, 1, 0, 1, 1e-1, 1.0),         # smallest legal problem
    (250, 4, 10, 2, 1e-3, 12.0),     # P does not divide N (R14): slices of 62, 63, 62, 63
    (500, 7, 20, 3, 1e-3, 16.0),     # slices of 71 / 72, M = 112, tiles straddle uneven slice boundaries
    (64, 64, 3, 1, 1e-3, 4.0),       # one eigenpair per slice
    (48, 48, 0, 2, 1e-3, 4.0),       # M = 1: every submatrix is one diagonal entry
    (255, 5, 8, 2, 1e-3, 12.0),      # odd N: the library works on a leading dimension of N + 1 internally (m = 51, M = 67)
    (1001, 7, 20, 3, 1e-3, 16.0),    # odd N, several 128-tiles, m = 143, M = 183
    (3, 1, 0, 1, 1e-1, 1.0),         # smallest odd problem
    (66, 64, 2, 2, 1e-3, 4.0),       # slices of 1 and 2
]


@pytest.mark.parametrize("route", [0, 1])   # 0 = the library's choice (tridiagonal route from M = 16 on), 1 = the Jacobi kernels
@pytest.mark.parametrize("N,P,w,iters,amp,width", SMALL_CASES)
def test_stepwise_parity_small(N, P, w, iters, amp, width, route, monkeypatch):
    monkeypatch.setitem(OPTS, "step2_route", route)
    p = gen.small_problem(N, amp, width, seed=1000 + N)
    nF = p.normF
    # step 2: shifts and zero-padded start vectors
    g2 = gpu_solve(p.A, P, w, iters, p.alpha, last_step=2)
    V2, eps, info2 = oracle.step2(p.A, P, w)
    assert g2["info"] == 0 and info2 == 0
    assert np.abs(g2["eps"] - eps).max() <= 1e-13 * max(1.0, nF)
    assert np.array_equal(g2["Vr"] == 0.0, V2 == 0.0) or np.abs(align_signs(g2["Vr"], V2) - V2).max() < 1e-9
    M, g0, lo, off = oracle.partition(N, P, w)
    cnt = oracle.slice_counts(N, P)
    for s in range(P):   # exactly zero outside the slice's window
        rows = g2["Vr"][g0[s]:g0[s] + cnt[s]]
        mask = np.ones(N, bool)
        mask[lo[s]:lo[s] + M] = False
        assert np.all(rows[:, mask] == 0.0)
    assert np.abs(align_signs(g2["Vr"], V2) - V2).max() < 1e-9
    # step 3 (Eq. 11) from the ORACLE's start vectors' signs
    g3 = gpu_solve(p.A, P, w, iters, p.alpha, last_step=3)
    V3 = oracle.step3(p.A, V2, eps, iters, p.alpha)
    assert np.abs(align_signs(g3["Vr"], V3) - V3).max() < 1e-9
    # step 4 (Gram-Schmidt as Cholesky-QR) and step 5
    g = gpu_solve(p.A, P, w, iters, p.alpha)
    o = oracle.pfsm(p.A, P, w, iters, p.alpha)
    check_gates(p.A, g, o)
    assert np.abs(align_signs(g["Vr"], o["Vr"]) - o["Vr"]).max() < 1e-8
    # uniqueness of thin QR: V_out^T V_in = R upper triangular with positive diagonal (reading R10)
    R = g["Vr"] @ g3["Vr"].T
    assert np.abs(np.tril(R, -1)).max() < 1e-10
    assert np.all(np.diag(R) > 0)


@pytest.mark.parametrize("N,P,w", [(256, 4, 16), (270, 6, 4), (600, 3, 20)])
def test_l2_resident_jacobi_fallback_matches_oracle(N, P, w, monkeypatch):
    # the L2-resident cluster kernel is the fallback for submatrices too large for shared memory; force it
    monkeypatch.setitem(OPTS, "step2_route", 1)      # (above M = 160 the tridiagonal route is the default)
    monkeypatch.setitem(OPTS, "jacobi_l2", 1)
    p = gen.small_problem(N, 1e-3, 12.0, seed=1000 + N)
    g2 = gpu_solve(p.A, P, w, 1, p.alpha, last_step=2)
    V2, eps, info2 = oracle.step2(p.A, P, w)
    assert g2["info"] == 0 and info2 == 0
    assert np.abs(g2["eps"] - eps).max() <= 1e-13 * max(1.0, p.normF)
    assert np.abs(align_signs(g2["Vr"], V2) - V2).max() < 1e-9


# step-2 routes of the wide-window regime: tridiagonalization with full symmetric storage (batch fits L2), lower-triangle
# storage (batch larger than L2) or blocked (dlatrd-style panels, read-only lower-triangle pass per column, one DMMA rank-2NB
# trailing update per panel), and the persistent-grid Jacobi
WIDE_ROUTES = [(("step2_route", 2),), (("step2_route", 2), ("sytrd_storage", 2)), (("step2_route", 3),),
               (("step2_route", 2), ("sytrd_storage", 3))]   # last: blocked tridiagonalization (panel + DMMA rank-2NB update)


@pytest.mark.parametrize("route", WIDE_ROUTES)
@pytest.mark.parametrize("N,P,w", [(256, 4, 16), (270, 6, 4), (600, 3, 20), (66, 64, 2), (96, 4, 100), (300, 200, 30)])
def test_wide_window_routes_forced_at_small_shapes_match_oracle(N, P, w, route, monkeypatch):
    # the two step-2 routes of the wide-window regime (M > 512), forced at shapes the oracle finishes quickly:
    # several slices per CTA, odd M, one-eigenpair slices, window >= N, more slices than co-resident CTAs
    for key, value in route:
        monkeypatch.setitem(OPTS, key, value)
    p = gen.small_problem(N, 1e-3, 12.0, seed=1000 + N)
    g2 = gpu_solve(p.A, P, w, 1, p.alpha, last_step=2)
    V2, eps, info2 = oracle_step2_memo(p.A, P, w)
    assert g2["info"] == 0 and info2 == 0
    assert np.abs(g2["eps"] - eps).max() <= 1e-13 * max(1.0, p.normF)
    assert np.abs(align_signs(g2["Vr"], V2) - V2).max() < 1e-9
    again = gpu_solve(p.A, P, w, 1, p.alpha, last_step=2)      # fixed operation and reduction order: same bits
    assert np.array_equal(again["Vr"], g2["Vr"]) and np.array_equal(again["eps"], g2["eps"])


@pytest.mark.parametrize("route", WIDE_ROUTES)
@pytest.mark.parametrize("N,P,w,iters", [(1200, 2, 0, 1), (1280, 4, 200, 2), (1102, 2, 1, 1)])
def test_wide_windows_beyond_512_match_oracle(N, P, w, iters, route, monkeypatch):
    # M = 600, 720 (gamma = 0.56) and 553 (odd); full solve against the oracle
    for key, value in route:                            # (the tridiagonal route is the default beyond M = 160)
        monkeypatch.setitem(OPTS, key, value)
    p = gen.small_problem(N, 1e-3, 24.0, seed=5000 + N + w)
    g2 = gpu_solve(p.A, P, w, iters, p.alpha, last_step=2)
    V2, eps, info2 = oracle_step2_memo(p.A, P, w)
    assert g2["info"] == 0 and info2 == 0
    assert np.abs(g2["eps"] - eps).max() <= 1e-12 * max(1.0, p.normF)
    assert np.abs(align_signs(g2["Vr"], V2) - V2).max() < 1e-8
    g = gpu_solve(p.A, P, w, iters, p.alpha)
    o = oracle_pfsm_memo(p.A, P, w, iters, p.alpha)
    check_gates(p.A, g, o)


@pytest.mark.parametrize("route", WIDE_ROUTES)
def test_wide_window_routes_on_doubly_degenerate_spectrum(route, monkeypatch):
    # A = blockdiag(B, B): every eigenvalue is exactly double.  The eigenvectors of a pair are not unique, so only
    # rotation-invariant quantities are compared (reading R16); the tridiagonal route has no re-orthogonalization
    # inside clusters (reading R25) and must still hand step 4 independent vectors (info = 0)
    for key, value in route:
        monkeypatch.setitem(OPTS, key, value)
    n = 96
    B = gen.small_problem(n, 5e-2, 8.0, seed=4242).A
    A = np.zeros((2 * n, 2 * n))
    A[:n, :n] = B
    A[n:, n:] = B
    ex = np.linalg.eigvalsh(A)
    alpha = 0.5 / np.abs(ex).max() ** 2
    for P, w in [(1, 0), (2, 2 * n)]:                   # M = N: every slice sees the whole (degenerate) spectrum
        g2 = gpu_solve(A, P, w, 2, alpha, last_step=2)
        assert g2["info"] == 0
        assert np.abs(g2["eps"] - ex).max() < 1e-13 * np.linalg.norm(A)
        g = gpu_solve(A, P, w, 2, alpha)
        assert g["info"] == 0
        assert np.abs(g["lam"] - ex).max() < 1e-12 * np.linalg.norm(A)
        assert np.abs(g["Vr"] @ g["Vr"].T - np.eye(2 * n)).max() <= 1e-12 * 2 * n
        assert g["resid"].max() < 1e-11 * np.linalg.norm(A)


@pytest.mark.parametrize("storage", [0, 2, 3])
def test_tridiagonal_route_on_near_degenerate_gaps(storage, monkeypatch):
    # A = Q diag(d) Q^T with pairs of eigenvalues separated by RELATIVE gaps 1e-15 .. 1e-6: too close for inverse iteration
    # alone (two vectors of a pair come out nearly parallel and step 4 would orthonormalize noise), not exactly equal.
    # The cluster pass (re-orthogonalization + re-iteration below 1e-7 ||T||, LAPACK dstein's scheme) must hand step 4
    # well-conditioned vectors: info = 0, eigenvalues and residuals to rounding, for every tridiagonalization kernel.
    monkeypatch.setitem(OPTS, "step2_route", 2)
    monkeypatch.setitem(OPTS, "sytrd_storage", storage)
    gaps = [1e-15, 1e-14, 1e-13, 1e-12, 1e-11, 1e-10, 1e-9, 1e-8, 1e-7, 1e-6]
    base = np.linspace(-1.0, 1.0, 120)
    d = np.concatenate([base] + [[base[7 * q + 3] * (1.0 + gp) + (gp if base[7 * q + 3] == 0 else 0.0)] for q, gp in enumerate(gaps)])
    d = np.sort(d)
    N = d.size
    assert N % 2 == 0
    Q = gen.householder_orthogonal(N, 8, seed=77)
    A = Q @ np.diag(d) @ Q.T
    A = 0.5 * (A + A.T)
    nA = np.linalg.norm(A)
    alpha = 0.5 / np.abs(d).max() ** 2
    for P, w in [(1, 0), (2, N)]:                       # M = N: every slice sees all the close pairs
        g2 = gpu_solve(A, P, w, 1, alpha, last_step=2)
        assert g2["info"] == 0
        assert np.abs(g2["eps"] - d).max() < 1e-13 * nA
        Y = g2["Vr"]
        assert np.abs(Y @ Y.T - np.eye(N)).max() < 1e-7     # close pairs included: the cluster pass orthogonalized them
        assert np.abs(Y @ A - g2["eps"][:, None] * Y).max() < 1e-12 * nA
        g = gpu_solve(A, P, w, 1, alpha)
        assert g["info"] == 0
        assert np.abs(g["lam"] - d).max() < 1e-12 * nA
        assert np.abs(g["Vr"] @ g["Vr"].T - np.eye(N)).max() <= 1e-12 * N
        assert g["resid"].max() < 1e-11 * nA


@pytest.mark.parametrize("n", [1100, 2100])
def test_cluster_pass_on_exact_doubles_at_large_submatrix_orders(n):
    # A = blockdiag(B, B), P = 1: one submatrix of order M = 2n whose every eigenvalue is exactly double, so EVERY vector
    # goes through the re-orthogonalization pass (reading R25) -- with its solves staged in shared memory as a whole
    # (M = 2200) and in chunks (M = 4200 > 4096).  Property-checked (the oracle's Jacobi would need far too long): eigenvalues vs
    # LAPACK on B, residuals, and orthonormality of the start vectors themselves, pairs included.
    B = gen.small_problem(n, 1e-3, 24.0, seed=4300 + n).A
    N = 2 * n
    A = np.zeros((N, N))
    A[:n, :n] = B
    A[n:, n:] = B
    mu = np.repeat(np.linalg.eigvalsh(B), 2)
    nA = np.linalg.norm(A)
    g2 = gpu_solve(A, 1, 0, 1, 0.5 / np.abs(mu).max() ** 2, last_step=2)
    assert g2["info"] == 0
    assert np.abs(g2["eps"] - mu).max() <= 1e-12 * nA
    Y = torch.from_numpy(g2["Vr"]).cuda()
    dA = torch.from_numpy(A).cuda()
    R = Y @ dA - torch.from_numpy(g2["eps"]).cuda()[:, None] * Y
    assert R.abs().max().item() <= 1e-12 * nA
    assert (Y @ Y.T - torch.eye(N, dtype=torch.float64, device="cuda")).abs().max().item() < 1e-7


@pytest.mark.parametrize("mult", [3, 13])
def test_tridiagonal_route_on_exact_multiplets(mult):
    # A = Q diag(d) Q^T with every eigenvalue repeated `mult` times (13 = the multiplet size of BASELINE config 2,
    # here exactly degenerate up to rounding): inverse iteration has no re-orthogonalization inside clusters (reading
    # R25), so the vectors of a multiplet come out as independent random combinations and step 4 must make them
    # orthonormal.  Only rotation-invariant quantities are compared (reading R16).  P = 2 with full windows: M = N > 160.
    nm = 20
    N = nm * mult
    if N % 2:
        N += mult
        nm += 1
    d = np.repeat(np.linspace(-1.0, 1.0, nm), mult)
    Q = gen.householder_orthogonal(N, 6, seed=99)
    A = (Q * d) @ Q.T
    A = 0.5 * (A + A.T)
    nF = np.linalg.norm(A)
    g2 = gpu_solve(A, 2, N, 2, 0.5, last_step=2)
    assert g2["info"] == 0
    assert np.abs(g2["eps"] - d).max() < 1e-13 * nF
    g = gpu_solve(A, 2, N, 2, 0.5)
    assert g["info"] == 0
    assert np.abs(g["lam"] - d).max() < 1e-12 * nF
    assert np.abs(g["Vr"] @ g["Vr"].T - np.eye(N)).max() <= 1e-12 * N
    assert g["resid"].max() < 1e-11 * nF


@pytest.mark.parametrize("N", [3000, 4096, 5000, 8192])
def test_submatrix_order_up_to_the_library_limit(N):
    # P = 1: the submatrix is A itself, M = N = 3000 ("M <= 3000"), 4096 (the largest order the full-storage,
    # blocked and persistent-grid-Jacobi kernels take), 5000 and 8192 (the library limit: the lower-triangle
    # tridiagonalization and 24-32 rows per thread in the back-transformation).  PROPERTY-checked, not oracle-checked: the
    # oracle's Jacobi would need hours, so step 2 is held to its definition -- eigenvalues vs LAPACK, residuals, orthonormality
    p = gen.small_problem(N, 1e-3, 48.0, seed=6000 + N)
    g2 = gpu_solve(p.A, 1, 0, 1, p.alpha, last_step=2)
    assert g2["info"] == 0
    dA = torch.from_numpy(p.A).cuda()
    mu = torch.linalg.eigvalsh(dA).cpu().numpy()
    assert np.abs(g2["eps"] - mu).max() <= 1e-12 * p.normF
    Y = torch.from_numpy(g2["Vr"]).cuda()
    R = Y @ dA - torch.from_numpy(g2["eps"]).cuda()[:, None] * Y
    assert R.abs().max().item() <= 1e-12 * p.normF
    assert (Y @ Y.T - torch.eye(N, dtype=torch.float64, device="cuda")).abs().max().item() < 1e-7   # eps ||A|| / gap (R25)


def test_iters_zero_is_gram_schmidt_of_start_vectors():
    p = gen.small_problem(288, 1e-3, 16.0, seed=77)
    g = gpu_solve(p.A, 4, 12, 0, p.alpha)
    o = oracle.pfsm(p.A, 4, 12, 0, p.alpha)
    check_gates(p.A, g, o)


def test_diagonal_input_is_a_fixed_point():
    # P1: B_s diagonal -> eps = d, start vectors = unit vectors, every step leaves them unchanged
    N = 384
    d = np.sort(gen.uniform(5, gen.STREAM_TEST, 0, N) * 2 - 1)
    g = gpu_solve(np.diag(d), 3, 20, 3, 0.5)
    assert g["info"] == 0
    assert np.abs(g["lam"] - d).max() < 1e-14
    assert np.abs(np.abs(g["Vr"]) - np.eye(N)).max() < 1e-14
    assert g["resid"].max() < 1e-14


def test_exact_degeneracy_invariants_only():
    N = 256
    d = np.repeat(np.arange(N // 8, dtype=np.float64) * 0.1, 8)
    g = gpu_solve(np.diag(d), 4, 16, 2, 0.5 / d.max() ** 2)
    assert g["info"] == 0
    np.testing.assert_allclose(np.sort(g["lam"]), d, atol=1e-13)
    assert np.abs(g["Vr"] @ g["Vr"].T - np.eye(N)).max() < 1e-12 * N
    assert g["resid"].max() < 1e-13


def test_block_diagonal_slices_exact():
    # P2 on the GPU: blocks = slices with separated spectra -> PFSM exact, incl. clamped end windows
    P, m, w = 4, 64, 16
    N = P * m
    A = np.zeros((N, N))
    expected = []
    for s in range(P):
        d = 10.0 * s + np.sort(gen.uniform(77, gen.STREAM_TEST, 100 * s, m))
        Q = gen.householder_orthogonal(m, 2, 300 + s)
        Bs = (Q * d) @ Q.T
        Bs = 0.5 * (Bs + Bs.T)
        A[s * m:(s + 1) * m, s * m:(s + 1) * m] = Bs
        expected.append(np.linalg.eigvalsh(Bs))
    expected = np.concatenate(expected)
    g = gpu_solve(A, P, w, 2, 0.5 / 31.0 ** 2)
    nA = np.linalg.norm(A)
    assert g["info"] == 0
    np.testing.assert_allclose(g["lam"], expected, atol=1e-13 * nA)
    assert g["resid"].max() < 1e-13 * nA


def test_breakdown_is_flagged_for_dependent_vectors():
    # P12 / PAPER.md:98: A = Q D Q^T with a dense random Q.  The GPU must either flag it (info != 0)
    # or return residuals far above the well-conditioned case -- never silently "succeed".
    N, P, w = 256, 4, 8
    d = np.sort(gen.uniform(51, gen.STREAM_TEST, 0, N) * 2 - 1)
    X = gen.normal(51, gen.STREAM_TEST, 10_000, N * N).reshape(N, N)
    Q, _ = np.linalg.qr(X)
    A = (Q * d) @ Q.T
    A = 0.5 * (A + A.T)
    g = gpu_solve(A, P, w, 3, 0.5)
    good = gen.small_problem(N, 1e-3, 8.0, seed=51)
    gg = gpu_solve(good.A, P, w, 3, good.alpha)
    assert gg["info"] == 0
    assert g["info"] != 0 or g["resid"].max() > 100 * gg["resid"].max()


@pytest.mark.parametrize("group", [2, 4])
def test_step4_panel_groups_match_gram_schmidt(group):
    # step 4 at a size with a tail: N = 3700 = 28 full panels + 116 columns, so with groups of 4 the schedule mixes groups of
    # four panels (K = 512 trailing updates, inner updates with K = 128, 256, 384), pairs and a ragged last panel; both
    # groupings must deliver THE Gram-Schmidt basis (uniqueness of QR), checked against the oracle on a leading block of columns
    N = 3700
    X = gen.normal(23, gen.STREAM_TEST, 0, N * N).reshape(N, N) + 4 * np.sqrt(N) * np.eye(N)
    h = pfsm.Handle(N, 1, 0, 0, 1.0, options={"cholesky_group": group})
    dV = dev(X)
    h.orthonormalize(dV)
    assert h.info() == 0
    Vg = dV.cpu().numpy()
    dVg = torch.from_numpy(Vg).cuda()
    assert (dVg @ dVg.T - torch.eye(N, dtype=torch.float64, device="cuda")).abs().max().item() <= 1e-12 * N
    R = dVg @ dev(X).T                                        # V_out^T X = R: upper triangular, positive diagonal
    assert torch.tril(R, -1).abs().max().item() < 1e-9 * np.sqrt(N) * 4
    assert (torch.diagonal(R) > 0).all()
    ncol = 300
    Vo, info = oracle.step4_mgs(X, ncol)                      # Gram-Schmidt of the first columns does not depend on the rest
    assert info == 0
    assert np.abs(Vg[:ncol] - Vo[:ncol]).max() < 1e-12
    h.destroy()


@pytest.mark.parametrize("N", [64, 200, 258, 384, 131, 257])   # (odd N: staged through a padded copy)
def test_step4_alone_matches_gram_schmidt(N):
    # step 4 on arbitrary (well-conditioned) vectors: Cholesky-QR == modified Gram-Schmidt (uniqueness of
    # thin QR with positive diagonal R, reading R10 / pin P11)
    X = gen.normal(17, gen.STREAM_TEST, 0, N * N).reshape(N, N) + 4 * np.sqrt(N) * np.eye(N)
    h = pfsm.Handle(N, 1, 0, 0, 1.0)
    dV = dev(X)
    h.orthonormalize(dV)
    assert h.info() == 0
    Vo, info = oracle.step4_mgs(X)
    assert info == 0
    Vg = dV.cpu().numpy()
    assert np.abs(Vg - Vo).max() < 1e-12
    assert np.abs(Vg @ Vg.T - np.eye(N)).max() <= 1e-12 * N
    h.destroy()


def test_step4_flags_dependent_vectors():
    # P12: a duplicated vector makes V^T V singular: both sides must flag it, at the second copy
    N = 256
    X = gen.normal(18, gen.STREAM_TEST, 0, N * N).reshape(N, N) + 4 * np.sqrt(N) * np.eye(N)
    X[200] = X[131]
    _, info_o = oracle.step4_mgs(X)
    h = pfsm.Handle(N, 1, 0, 0, 1.0)
    dV = dev(X)
    h.orthonormalize(dV)
    assert info_o == 201
    assert h.info() == 201
    # and the flag is cleared by the next healthy call
    X[200] = gen.normal(19, gen.STREAM_TEST, 0, N)
    dV = dev(X)
    h.orthonormalize(dV)
    assert h.info() == 0
    h.destroy()


@pytest.mark.parametrize("N", [320, 321])
def test_step5_alone_matches_definition(N):
    p = gen.small_problem(N, 0.05, 10.0, seed=33)
    X = gen.normal(19, gen.STREAM_TEST, 0, N * N).reshape(N, N)
    X /= np.linalg.norm(X, axis=1, keepdims=True)
    h = pfsm.Handle(N, 1, 0, 0, 1.0)
    dl = torch.empty(N, dtype=torch.float64, device="cuda")
    h.rayleigh(dev(p.A), dev(X), dl)
    lam_o, res_o = oracle.step5(p.A, X)
    assert np.abs(dl.cpu().numpy() - lam_o).max() < 1e-13
    assert np.abs(h.residuals().cpu().numpy() - res_o).max() < 1e-13
    h.destroy()


def test_solve_is_deterministic_and_ignores_v_input():
    p = gen.problem(0)
    c = p.cfg
    a = gpu_solve(p.A, c.P, c.window, c.iters, p.alpha)
    b = gpu_solve(p.A, c.P, c.window, c.iters, p.alpha)
    assert np.array_equal(a["lam"], b["lam"]) and np.array_equal(a["Vr"], b["Vr"])


@pytest.mark.parametrize("case", ["config0", "config1", "wide", "odd"])
def test_host_buffer_entry_point_matches_device_entry_point(case):
    # config 0: shared-memory Jacobi, config 1: tridiagonal route -- both with the diagonal blocks uploaded ahead of A;
    # wide: M = 700 (blocks as large as A: plain upload)
    if case == "wide":
        p = gen.small_problem(1000, 1e-3, 24.0, seed=808)
        N, P, w, iters = 1000, 2, 100, 2
    elif case == "odd":
        p = gen.small_problem(777, 1e-3, 24.0, seed=809)
        N, P, w, iters = 777, 7, 20, 2
    else:
        p = gen.problem(int(case[-1]))
        N, P, w, iters = p.cfg.N, p.cfg.P, p.cfg.window, p.cfg.iters
    h = pfsm.Handle(N, P, w, iters, p.alpha)
    Ah = torch.from_numpy(p.A).pin_memory()
    Vh = torch.empty((N, N), dtype=torch.float64).pin_memory()
    lh = torch.empty((N,), dtype=torch.float64).pin_memory()
    h.solve_host(Ah, Vh, lh)
    torch.cuda.synchronize()
    assert h.info() == 0
    ref = gpu_solve(p.A, P, w, iters, p.alpha)
    assert np.array_equal(lh.numpy(), ref["lam"]) and np.array_equal(Vh.numpy(), ref["Vr"])
    # A = A^T: only the lower block triangle (256-row blocks) and the P diagonal submatrices (entries with
    # |row - col| < M) are read from the host buffer and cross PCIe
    M = min(N, -(-N // P) + 2 * w)
    rr, cc = np.meshgrid(np.arange(N), np.arange(N), indexing="ij")
    unread = (cc >= (rr // 256 + 1) * 256) & (cc - rr >= M)
    Ah.numpy()[unread] = float("nan")
    Vh.zero_()
    lh.zero_()
    h.solve_host(Ah, Vh, lh)
    torch.cuda.synchronize()
    assert np.array_equal(lh.numpy(), ref["lam"]) and np.array_equal(Vh.numpy(), ref["Vr"])
    h.destroy()


def test_solve_on_a_side_stream():
    p = gen.problem(0)
    c = p.cfg
    N = c.N
    st = torch.cuda.Stream()
    h = pfsm.Handle(N, c.P, c.window, c.iters, p.alpha)
    dA = dev(p.A)
    dV = torch.empty((N, N), dtype=torch.float64, device="cuda")
    dl = torch.empty((N,), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    with torch.cuda.stream(st):
        h.solve(dA, dV, dl, stream=st)
    assert h.info(stream=st) == 0
    ref = gpu_solve(p.A, c.P, c.window, c.iters, p.alpha)
    assert np.array_equal(dl.cpu().numpy(), ref["lam"])
    h.destroy()


def test_validity_guard_follows_the_paper_failure_mode():
    """PFSM is valid for diagonally dominant matrices; otherwise standard diagonalization is used.
    The guard must pass a dominant matrix, and flag A = Q D Q^T with a dense random Q (no dominance: the submatrix
    eigenvectors say nothing about A's), where the oracle shows the same large residuals."""
    N, P, w, iters = 256, 4, 16, 3
    p = gen.small_problem(N, 1e-3, 16.0, seed=77)
    nF = p.normF
    h = pfsm.Handle(N, P, w, iters, p.alpha)
    dV = torch.empty((N, N), dtype=torch.float64, device="cuda")
    dl = torch.empty((N,), dtype=torch.float64, device="cuda")
    h.solve(dev(p.A), dV, dl)
    use_std, mx, info = h.check_validity(1e-2 * nF)
    r = h.residuals().cpu().numpy()
    assert not use_std and info == 0 and mx == r.max()
    assert h.check_validity(0.5 * r.max())[0]                      # same solve, tighter tolerance: flagged
    Q = gen.householder_orthogonal(N, N // 2, seed=5)
    A2 = Q @ np.diag(p.d) @ Q.T
    A2 = 0.5 * (A2 + A2.T)
    h.solve(dev(A2), dV, dl)
    use_std, mx2, info2 = h.check_validity(1e-2 * nF)
    o = oracle.pfsm(A2, P, w, iters, p.alpha)
    assert o["info"] != 0 or o["resid"].max() > 1e-2 * nF           # the oracle shows the failure too
    assert use_std and (info2 != 0 or mx2 > 1e-2 * nF)
    with pytest.raises(pfsm.PfsmError):
        h.check_validity(float("nan"))
    h.destroy()


@pytest.mark.parametrize("N,P,w,iters", [(2048, 16, 32, 3), (600, 3, 20, 2), (1000, 7, 30, 4)])
def test_chained_launches_change_no_bit(N, P, w, iters, monkeypatch):
    """The step-3 GEMMs (and step 4's Gram product) overlap their last waves through programmatic dependent launch and
    per-row-block counters.  That is scheduling only: the result must equal the plain stream-ordered
    launches bit for bit, solve after solve (a tile that started before its operand rows were complete would differ)."""
    p = gen.small_problem(N, 1e-3, 24.0, seed=52000 + N)
    chained = [gpu_solve(p.A, P, w, iters, p.alpha) for _ in range(3)]
    monkeypatch.setitem(OPTS, "chain_launches", 0)
    plain = gpu_solve(p.A, P, w, iters, p.alpha)
    for g in chained:
        assert g["info"] == 0
        assert np.array_equal(g["Vr"], plain["Vr"]) and np.array_equal(g["lam"], plain["lam"])
        assert np.array_equal(g["resid"], plain["resid"])


@pytest.mark.parametrize("k,family", [(0, "default"), (1, "default"), (2, "default"), (5, "default"),
                                      (0, "jacobi"), (1, "jacobi"), (2, "jacobi"), (5, "jacobi")])
def test_baseline_configs_full_oracle(k, family, monkeypatch):
    """BASELINE.json configs 0-2 at full size, and the Cu256-shaped extra case (N = 1664, window at the paper's
    gamma = 0.25: M = 416, clamped windows on 4 of 13 slices): element-by-element gates against the full oracle run.
    default = the route the library picks (tridiagonalization, submatrices resident in the clusters' distributed shared
    memory); the Jacobi family is forced as well."""
    if family != "default":
        monkeypatch.setitem(OPTS, "step2_route", 1 if family == "jacobi" else 2)
    p = gen.problem(k)
    c = p.cfg
    g = gpu_solve(p.A, c.P, c.window, c.iters, p.alpha)
    o = oracle_pfsm_memo(p.A, c.P, c.window, c.iters, p.alpha)
    check_gates(p.A, g, o)
    assert np.abs(g["eps"] - o["eps"]).max() <= 1e-12 * p.normF


def _check_steps_4_5_at_full_size(p, g3, g, k):
    """Step 4 through the uniqueness of QR, step 5 on sampled columns the oracle computes one by one, trace and
    residual enclosure -- properties that hold at any size."""
    c = p.cfg
    N, m = c.N, c.m
    nF = p.normF
    assert g["info"] == 0
    Vg = torch.from_numpy(g["Vr"]).cuda()
    V3g = torch.from_numpy(g3["Vr"]).cuda()
    eye_err = (Vg @ Vg.T - torch.eye(N, dtype=torch.float64, device="cuda")).abs().max().item()
    assert eye_err <= 1e-12 * N
    R = Vg @ V3g.T
    assert torch.tril(R, -1).abs().max().item() < 1e-9
    assert (torch.diagonal(R) > 0).all()
    cols = [0, 1, m - 1, m, N // 2, N - 2, N - 1] + [int(x) for x in (gen.uniform(9, gen.STREAM_TEST, k, 9) * N)]
    for i in cols:
        lam_o, res_o = oracle.step5(p.A, g["Vr"], i, i + 1)
        assert abs(lam_o[i] - g["lam"][i]) <= 1e-10 * nF
        assert abs(res_o[i] - g["resid"][i]) <= 1e-9 * nF
    assert abs(g["lam"].sum() - np.trace(p.A)) <= 1e-9
    ex = torch.linalg.eigvalsh(torch.from_numpy(p.A).cuda()).cpu().numpy()   # comparison only (P9 enclosure)
    idx = np.searchsorted(ex, g["lam"])
    near = np.minimum(np.abs(ex[np.clip(idx, 0, N - 1)] - g["lam"]), np.abs(ex[np.clip(idx - 1, 0, N - 1)] - g["lam"]))
    assert np.all(near <= g["resid"] + 1e-10)


def test_wide_window_config6_at_full_size():
    """Config 4's matrix at the paper's gamma = 0.25 (N = 8192, P = 16, M = 2048: the tridiagonalization route of
    step 2, lower-triangle storage).  The oracle's Jacobi needs minutes per 2048 x 2048 slice, so step 2 is checked
    against what it must deliver by definition -- the eigenpairs of rank off .. off+m-1 of B_s:
    eigenvalues against LAPACK on sampled slices, residuals ||B y - mu y||, zero padding -- and steps 4-5 as for
    configs 3-4."""
    p = gen.problem(6)
    c = p.cfg
    N, m = c.N, c.m
    g3 = gpu_solve(p.A, c.P, c.window, c.iters, p.alpha, last_step=2)
    assert g3["info"] == 0
    M, g0, lo, off = oracle.partition(N, c.P, c.window)
    assert M == 2048
    for s in (0, c.P // 2, c.P - 1):
        B = p.A[lo[s]:lo[s] + M, lo[s]:lo[s] + M]
        mu = np.linalg.eigvalsh(B)[off[s]:off[s] + m]
        eps_s = g3["eps"][g0[s]:g0[s] + m]
        assert np.abs(eps_s - mu).max() <= 1e-12 * p.normF
        rows = g3["Vr"][g0[s]:g0[s] + m]
        mask = np.ones(N, bool)
        mask[lo[s]:lo[s] + M] = False
        assert np.all(rows[:, mask] == 0.0)
        Y = rows[:, lo[s]:lo[s] + M]
        assert np.abs(Y @ B - eps_s[:, None] * Y).max() <= 1e-12 * np.linalg.norm(B)
        assert np.abs(np.einsum("ij,ij->i", Y, Y) - 1.0).max() < 1e-13
        assert np.abs(Y @ Y.T - np.eye(m)).max() < 1e-7     # eps ||B|| / gap; step 4 orthonormalizes (reading R25)
        if os.environ.get("PFSM_FULL_ORACLE") == "1" and s == c.P // 2:   # the oracle's own Jacobi: ~7 min on 16 cores
            mu_o, Y_o, sw = oracle.jacobi_eig(B)
            assert sw > 0
            assert np.abs(eps_s - mu_o[off[s]:off[s] + m]).max() <= 1e-12 * p.normF
            Yo = Y_o[:, off[s]:off[s] + m].T
            assert np.abs(align_signs(Y, Yo) - Yo).max() < 1e-7
    g3 = gpu_solve(p.A, c.P, c.window, c.iters, p.alpha, last_step=3)
    g = gpu_solve(p.A, c.P, c.window, c.iters, p.alpha)
    _check_steps_4_5_at_full_size(p, g3, g, 6)


def load_golden_large(k):
    """tests/golden/config{k}_oracle.txt (+ _vectors.npz): the full oracle run of config k, every index, written by
    tests/golden/make_golden_large.py from oracle/ + pfsm_inputs/ only."""
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    head, rows = {}, []
    for ln in open(os.path.join(here, f"config{k}_oracle.txt")):
        if ln.startswith("#"):
            continue
        f = ln.split()
        if len(f) == 2:
            head[f[0]] = float(f[1])
        elif len(f) == 3:
            rows.append([float(x) for x in f])
    arr = np.array(rows)
    vec = np.load(os.path.join(here, f"config{k}_oracle_vectors.npz"))
    return head, dict(lam=arr[:, 0], resid=arr[:, 1], eps=arr[:, 2], idx=vec["idx"], Vr=vec["Vr"])


@pytest.mark.parametrize("k,family", [(3, "default"), (3, "jacobi"), (4, "default"), (4, "jacobi")])
def test_baseline_configs_large_all_indices(k, family, monkeypatch):
    """BASELINE.json configs 3-4 (config 4 = bench.py's headline workload) at full size, in bench.py's launch
    configuration, against the FULL oracle run on EVERY index: the oracle's lambda, residuals and shifts for all N
    eigenpairs come from tests/golden/config{k}_oracle.txt (the oracle needs ~1e13 flop per config: minutes, so its
    output is stored by tests/golden/make_golden_large.py, which calls only oracle/ and pfsm_inputs/).  Gates are
    north_star's, per index.  On top: steps 2-3 against the live oracle on sampled whole slices (slices are
    independent), whole eigenvectors against the stored oracle vectors (sign-aligned), step 4 through the
    uniqueness of QR, trace and residual enclosure.  default = the tridiagonal route of step 2; jacobi = the
    shared-memory Jacobi (clusters of 8 half CTAs)."""
    if family == "jacobi":
        monkeypatch.setitem(OPTS, "step2_route", 1)
    p = gen.problem(k)
    c = p.cfg
    N, m = c.N, c.m
    nF = p.normF
    head, gold = load_golden_large(k)
    # the stored run is of THIS matrix and these parameters
    assert int(head["N"]) == N and head["alpha"] == p.alpha and abs(head["normF"] - nF) <= 1e-12 * nF
    assert head["ortho_max"] <= 1e-12 * N                                  # the oracle's own orthonormality gate
    g3 = gpu_solve(p.A, c.P, c.window, c.iters, p.alpha, last_step=3)
    assert g3["info"] == 0
    assert np.abs(g3["eps"] - gold["eps"]).max() <= 1e-12 * nF             # every shift (step 2, all slices)
    M, g0, lo, off = oracle.partition(N, c.P, c.window)
    for s in sorted({0, 1, c.P // 2, c.P - 1}):
        B = p.A[lo[s]:lo[s] + M, lo[s]:lo[s] + M]
        mu, Y, sw = oracle.jacobi_eig(B)
        assert sw > 0
        eps_s = mu[off[s]:off[s] + m]
        assert np.abs(g3["eps"][g0[s]:g0[s] + m] - eps_s).max() <= 1e-12 * nF
        V0 = np.zeros((N, N))
        V0[g0[s]:g0[s] + m, lo[s]:lo[s] + M] = Y[:, off[s]:off[s] + m].T
        eps_full = np.zeros(N)
        eps_full[g0[s]:g0[s] + m] = eps_s
        V3 = oracle.step3(p.A, V0, eps_full, c.iters, p.alpha, int(g0[s]), int(g0[s] + m))[g0[s]:g0[s] + m]
        Vg = g3["Vr"][g0[s]:g0[s] + m]
        assert np.abs(align_signs(Vg, V3) - V3).max() < 1e-8
    g = gpu_solve(p.A, c.P, c.window, c.iters, p.alpha)
    assert g["info"] == 0
    # ---- the north_star gates on all N indices, against the stored full oracle run
    assert np.abs(g["lam"] - gold["lam"]).max() <= 1e-10 * nF
    assert np.abs(g["resid"] - gold["resid"]).max() <= 1e-9 * nF
    assert np.abs(g["eps"] - gold["eps"]).max() <= 1e-12 * nF
    Vg = g["Vr"][gold["idx"]]
    assert np.abs(align_signs(Vg, gold["Vr"]) - gold["Vr"]).max() < 1e-7   # whole vectors after step 4 (cond(V) ~ 500 at config 4)
    _check_steps_4_5_at_full_size(p, g3, g, k)


# ------------------------------------------------------------------ row G: generalized variant A x = lambda S x
def gpu_generalized(A, S, P, w, iters, alpha):
    N = A.shape[0]
    h = pfsm.Handle(N, P, w, iters, alpha)
    dA, dS = dev(A), dev(S)
    dAp = torch.empty((N, N), dtype=torch.float64, device="cuda")
    h.generalized_reduce(dA, dS, dAp)
    info_r = h.info()
    dX = torch.empty((N, N), dtype=torch.float64, device="cuda")
    dl = torch.empty((N,), dtype=torch.float64, device="cuda")
    h.solve_generalized(dA, dS, dX, dl)
    out = dict(Ap=dAp.cpu().numpy(), Xr=dX.cpu().numpy(), lam=dl.cpu().numpy(), resid=h.residuals().cpu().numpy(),
               info=h.info(), info_reduce=info_r)
    h.destroy()
    return out


@pytest.mark.parametrize("N,P,w,iters", [(192, 4, 12, 2), (300, 5, 10, 3), (384, 3, 40, 2), (275, 5, 10, 2)])
def test_generalized_small_against_oracle(N, P, w, iters):
    p = gen.small_problem(N, 2e-3, 12.0, seed=600 + N)
    S = gen.banded_symmetric(N, np.ones(N), 1e-2, 6.0, 600 + N, gen.STREAM_S)
    g = gpu_generalized(p.A, S, P, w, iters, p.alpha)
    L, Ap, info = oracle.generalized_reduce(p.A, S)
    assert info == 0 and g["info"] == 0 and g["info_reduce"] == 0
    assert np.abs(g["Ap"] - Ap).max() < 1e-12 * max(1.0, np.abs(Ap).max())
    assert np.array_equal(g["Ap"], g["Ap"].T)                       # exactly symmetric
    o = oracle.pfsm(Ap, P, w, iters, p.alpha)
    Xo = oracle.generalized_back(L, o["Vr"])
    nF = float(np.linalg.norm(Ap))
    assert np.abs(g["lam"] - o["lam"]).max() <= 1e-10 * nF
    assert np.abs(g["resid"] - o["resid"]).max() <= 1e-9 * nF
    X = g["Xr"]
    assert np.abs(X @ S @ X.T - np.eye(N)).max() <= 1e-12 * N        # X^T S X = I (pin P13)
    assert np.abs(align_signs(X, Xo) - Xo).max() < 1e-8
    # generalized residual = L (A' v - lambda v): bounded by ||L|| r_i
    R = X @ p.A - (X @ S) * g["lam"][:, None]
    assert np.all(np.linalg.norm(R, axis=1) <= np.linalg.norm(L, 2) * g["resid"] + 1e-11)


def test_generalized_identity_overlap_equals_standard_path():
    p = gen.problem(0)
    c = p.cfg
    g = gpu_generalized(p.A, np.eye(c.N), c.P, c.window, c.iters, p.alpha)
    ref = gpu_solve(p.A, c.P, c.window, c.iters, p.alpha)
    assert np.array_equal(g["Ap"], p.A)
    assert np.array_equal(g["lam"], ref["lam"]) and np.array_equal(g["Xr"], ref["Vr"])


def test_generalized_flags_indefinite_overlap():
    N = 256
    p = gen.small_problem(N, 1e-3, 8.0, seed=71)
    S = np.eye(N)
    S[100, 100] = -1.0
    g = gpu_generalized(p.A, S, 4, 8, 1, p.alpha)
    assert g["info_reduce"] == 101 and g["info"] != 0


def test_generalized_config4g_properties():
    """BASELINE.json configs[4] generalized form at full size (N=8192).  The oracle's unblocked reduction needs
    ~1e12 flop in plain loops, so the reduction is pinned by properties that determine it uniquely: L lower
    triangular with positive diagonal and L L^T = S (uniqueness of Cholesky), L A' L^T = A; then the standard
    path on A' is the already-tested one, and X^T S X = I, A X = S X Lambda + L R hold for the result."""
    p = gen.problem(4, generalized=True)
    c = p.cfg
    N = c.N
    h = pfsm.Handle(N, c.P, c.window, c.iters, p.alpha)
    dA, dS = dev(p.A), dev(p.S)
    dAp = torch.empty((N, N), dtype=torch.float64, device="cuda")
    h.generalized_reduce(dA, dS, dAp)
    assert h.info() == 0
    Lt = torch.linalg.cholesky(dS)                       # comparison only: the unique factor
    back = Lt @ dAp @ Lt.T
    assert (back - dA).abs().max().item() < 1e-11
    assert (dAp - dAp.T).abs().max().item() == 0.0
    dX = torch.empty((N, N), dtype=torch.float64, device="cuda")
    dl = torch.empty((N,), dtype=torch.float64, device="cuda")
    h.solve_generalized(dA, dS, dX, dl)
    assert h.info() == 0
    eye_err = (dX @ dS @ dX.T - torch.eye(N, dtype=torch.float64, device="cuda")).abs().max().item()
    assert eye_err <= 1e-12 * N
    R = dX @ dA - (dX @ dS) * dl[:, None]
    rn = torch.linalg.norm(R, dim=1)
    res = h.residuals()
    assert bool((rn <= 1.01 * res + 1e-10).all())         # ||L|| <= 1.01 for S = I + 1e-4 perturbation
    # the standard path on A' gives the same eigenvalues
    dV = torch.empty((N, N), dtype=torch.float64, device="cuda")
    dl2 = torch.empty((N,), dtype=torch.float64, device="cuda")
    h.solve(dAp, dV, dl2)
    assert torch.equal(dl, dl2)
    h.destroy()


# ------------------------------------------------------------------ SCF-sequence mode (pfsm_solve_warm)
def gpu_warm(A, Vr_prev, P, w, iters, alpha):
    N = A.shape[0]
    h = pfsm.Handle(N, P, w, iters, alpha)
    dA, dV = dev(A), dev(Vr_prev)
    dl = torch.empty((N,), dtype=torch.float64, device="cuda")
    h.solve_warm(dA, dV, dl)
    out = dict(Vr=dV.cpu().numpy(), lam=dl.cpu().numpy(), resid=h.residuals().cpu().numpy(), info=h.info())
    h.destroy()
    return out


@pytest.mark.parametrize("N,P", [(384, 4), (384, 2), (385, 5)])    # M = 144, M = 240; odd N (M = 125)
def test_warm_start_sequence_matches_oracle(N, P):
    w, iters = 24, 3
    d = np.sort(gen.uniform(83, gen.STREAM_TEST, 0, N) * 2 - 1)
    X = gen.normal(83, gen.STREAM_TEST, 10_000, N * N).reshape(N, N)
    Q, _ = np.linalg.qr(X)
    A0 = (Q * d) @ Q.T
    A0 = 0.5 * (A0 + A0.T)
    dA = gen.normal(83, gen.STREAM_TEST, 500_000, N * N).reshape(N, N) * 5e-5
    dA = 0.5 * (dA + dA.T)
    _, V = np.linalg.eigh(A0)       # "standard diagonalization for the first SCF steps"
    Vg = Vo = V.T.copy()
    for k in range(1, 4):
        Ak = A0 + k * dA
        nF = float(np.linalg.norm(Ak))
        g = gpu_warm(Ak, Vg, P, w, iters, 0.5)
        o = oracle.pfsm_warm(Ak, Vo, P, w, iters, 0.5)
        assert g["info"] == 0 and o["info"] == 0
        assert np.abs(g["lam"] - o["lam"]).max() <= 1e-10 * nF
        assert np.abs(g["resid"] - o["resid"]).max() <= 1e-9 * nF
        assert np.abs(g["Vr"] @ g["Vr"].T - np.eye(N)).max() <= 1e-12 * N
        assert np.abs(align_signs(g["Vr"], o["Vr"]) - o["Vr"]).max() < 1e-8
        # residuals are those of (A_k, V): the change of basis is orthogonal
        R = g["Vr"] @ Ak - g["lam"][:, None] * g["Vr"]
        assert np.abs(np.linalg.norm(R, axis=1) - g["resid"]).max() < 1e-11
        Vg, Vo = g["Vr"], o["Vr"]


def test_warm_start_identity_basis_equals_plain_solve():
    p = gen.problem(0)
    c = p.cfg
    g = gpu_warm(p.A, np.eye(c.N), c.P, c.window, c.iters, p.alpha)
    ref = gpu_solve(p.A, c.P, c.window, c.iters, p.alpha)
    assert np.abs(g["lam"] - ref["lam"]).max() < 1e-14 and np.abs(g["Vr"] - ref["Vr"]).max() < 1e-13


@pytest.mark.parametrize("big", [False, True, "tridiag", "tridiag_grid"])
def test_solve_is_cuda_graph_capturable(big):
    # the whole solve enqueues kernels and memsets only (no host sync): capture once, replay many times.
    # big: N = 896 has 4 panel pairs, so step 4 runs its two-stream look-ahead schedule inside the capture.
    # tridiag: M = 256, step 2's tridiagonal route with one cluster per slice; tridiag_grid: M = 900, its persistent
    # cooperative grid (a cooperative launch inside the capture)
    if big == "tridiag":
        p = gen.small_problem(896, 1e-3, 16.0, seed=606)
        c = gen.Config(-1, "graph", 896, 4, 16, 2, 1e-3, 16.0)
    elif big == "tridiag_grid":
        p = gen.small_problem(1800, 1e-3, 16.0, seed=607)
        c = gen.Config(-1, "graph", 1800, 2, 0, 1, 1e-3, 16.0)
    elif big:
        p = gen.small_problem(896, 1e-3, 16.0, seed=606)
        c = gen.Config(-1, "graph", 896, 7, 16, 2, 1e-3, 16.0)
    else:
        p = gen.problem(0)
        c = p.cfg
    N = c.N
    h = pfsm.Handle(N, c.P, c.window, c.iters, p.alpha)
    dA = dev(p.A)
    dV = torch.empty((N, N), dtype=torch.float64, device="cuda")
    dl = torch.empty((N,), dtype=torch.float64, device="cuda")
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        h.solve(dA, dV, dl, stream=st)      # warm-up: one-time function attributes are set outside the capture
    st.synchronize()
    ref_l, ref_V = dl.clone(), dV.clone()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=st):
        h.solve(dA, dV, dl, stream=torch.cuda.current_stream())
    for _ in range(3):
        dV.fill_(float("nan"))
        dl.fill_(float("nan"))
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(dl, ref_l) and torch.equal(dV, ref_V)
    assert h.info() == 0
    h.destroy()


# ------------------------------------------------------------------ f2: the paper's Eq. 14-15 conversion
@pytest.mark.parametrize("N,niter", [(256, 1), (300, 3), (384, 6), (301, 3)])
def test_eq14_iteration_matches_oracle(N, niter):
    p = gen.small_problem(N, 2e-3, 12.0, seed=900 + N)
    B = gen.banded_symmetric(N, np.ones(N), 1e-2, 6.0, 900 + N, gen.STREAM_S)
    h = pfsm.Handle(N, 1, 0, 0, 1.0)
    dZ = torch.empty((N, N), dtype=torch.float64, device="cuda")
    h.standard_form_eq14(dev(p.A), dev(B), dZ, niter, symmetrize=False)
    Zg = dZ.cpu().numpy().T                     # column-major Z -> numpy Z[i, j]
    Zo = oracle.eq14_iteration(p.A, B, niter)
    assert np.abs(Zg - Zo).max() < 1e-13 * max(1.0, np.abs(Zo).max())
    h.standard_form_eq14(dev(p.A), dev(B), dZ, niter, symmetrize=True)
    Zs = dZ.cpu().numpy()
    assert np.array_equal(Zs, Zs.T)
    assert np.abs(Zs - oracle.eq14_iteration(p.A, B, niter, symmetrize=True)).max() < 1e-13
    h.destroy()


def test_eq14_converges_to_the_cholesky_route_on_config4g_shape():
    # both conversions feed the same standard eigenproblem when S is close to I: B^-1 A (symmetrized) and
    # L^-1 A L^-T have the same spectrum up to O(||S - I||^2) -- information, checked loosely
    N = 512
    p = gen.small_problem(N, 2e-3, 32.0, seed=77)
    S = gen.banded_symmetric(N, np.ones(N), 1e-4, 128.0, 77, gen.STREAM_S)
    h = pfsm.Handle(N, 4, 32, 2, p.alpha)
    dZ = torch.empty((N, N), dtype=torch.float64, device="cuda")
    h.standard_form_eq14(dev(p.A), dev(S), dZ, 8, symmetrize=False)
    Z = dZ.cpu().numpy().T
    assert np.abs(S @ Z - p.A).max() < 1e-14      # Eq. 15: B Z = A at convergence
    import scipy.linalg
    ex = scipy.linalg.eigh(p.A, S, eigvals_only=True)
    assert np.abs(np.sort(np.linalg.eigvals(Z).real) - ex).max() < 1e-10
    h.destroy()


# ------------------------------------------------------------------ seeded sweep over ragged shapes
def _fuzz_cases(count=24):
    u = gen.uniform(20260101, gen.STREAM_TEST, 0, 4 * count)
    cases = []
    for k in range(count):
        N = 2 * int(2 + u[4 * k] * 330)                      # even, 4 .. 662
        divs = [d for d in range(1, N + 1) if N % d == 0 and N // d >= 1]
        P = divs[int(u[4 * k + 1] * len(divs)) % len(divs)]
        if k % 3 == 2:
            P = 1 + int(u[4 * k + 1] * min(N, 40))           # any P: slices of unequal size (R14)
        m = -(-N // P)
        w = int(u[4 * k + 2] * 40)
        if min(N, m + 2 * w) > 512:                          # library limit on the submatrix order
            w = max(0, (512 - m) // 2)
        if m > 512:
            continue
        iters = int(u[4 * k + 3] * 4)
        cases.append((N, P, w, iters))
    return cases


@pytest.mark.parametrize("N,P,w,iters", _fuzz_cases())
def test_seeded_shape_sweep_against_oracle(N, P, w, iters):
    p = gen.small_problem(N, 1e-3, max(2.0, N / 16.0), seed=31000 + N + P)
    g = gpu_solve(p.A, P, w, iters, p.alpha)
    o = oracle.pfsm(p.A, P, w, iters, p.alpha)
    check_gates(p.A, g, o)
    assert np.abs(g["eps"] - o["eps"]).max() <= 1e-12 * max(1.0, p.normF)


def test_second_cholqr_pass_restores_orthogonality_of_ill_conditioned_vectors():
    # vectors with cond ~ 1e5: one Cholesky-QR pass leaves ~eps cond^2 ~ 1e-6 of non-orthogonality, two passes ~eps;
    # both are the Gram-Schmidt basis (same exact-arithmetic result, reading R10)
    N = 256
    Q1, _ = np.linalg.qr(gen.normal(41, gen.STREAM_TEST, 0, N * N).reshape(N, N))
    Q2, _ = np.linalg.qr(gen.normal(42, gen.STREAM_TEST, 0, N * N).reshape(N, N))
    X = (Q1 * np.logspace(0, -5, N)) @ Q2.T
    Vo, info = oracle.step4_mgs(X)
    assert info == 0
    h = pfsm.Handle(N, 1, 0, 0, 1.0)
    errs = {}
    for passes in (1, 2):
        h.set_cholqr_passes(passes)
        dV = dev(X)
        h.orthonormalize(dV)
        assert h.info() == 0
        Vg = dV.cpu().numpy()
        errs[passes] = np.abs(Vg @ Vg.T - np.eye(N)).max()
        if passes == 2:
            assert np.abs(Vg - Vo).max() < 1e-9       # MGS itself loses eps cond ~ 1e-11 here
    assert errs[2] < 1e-13 and errs[2] < 1e-3 * errs[1]
    h.destroy()


@pytest.mark.parametrize("family", ["default", "jacobi"])
@pytest.mark.parametrize("N,P,w", [(800, 2, 0), (1024, 2, 0), (1024, 4, 128)])
def test_large_submatrices_up_to_the_jacobi_limit(N, P, w, family, monkeypatch):
    # M = 400 and M = 512.  default: the tridiagonal route (cluster-barrier tridiagonalization); jacobi: the
    # shared-memory kernel with a cluster of 8 (M = 400) and the L2-resident fallback with 16 doubles/lane (M = 512)
    if family == "jacobi":
        monkeypatch.setitem(OPTS, "step2_route", 1)
    p = gen.small_problem(N, 1e-3, 24.0, seed=5000 + N + w)
    g2 = gpu_solve(p.A, P, w, 1, p.alpha, last_step=2)
    V2, eps, info2 = oracle_step2_memo(p.A, P, w)
    assert g2["info"] == 0 and info2 == 0
    assert np.abs(g2["eps"] - eps).max() <= 1e-12 * max(1.0, p.normF)
    assert np.abs(align_signs(g2["Vr"], V2) - V2).max() < 1e-8
    g = gpu_solve(p.A, P, w, 1, p.alpha)
    o = oracle_pfsm_memo(p.A, P, w, 1, p.alpha)
    check_gates(p.A, g, o)


@pytest.mark.parametrize("k,reps", [(0, 60), (1, 12), (2, 8)])
def test_repeated_solves_are_bitwise_identical(k, reps):
    # race detector: the cluster exchange of step 2, the two-stream schedule of step 4 and every reduction have a
    # fixed order, so a solve is bitwise reproducible; any data race shows up as a differing bit sooner or later
    p = gen.problem(k)
    c = p.cfg
    N = c.N
    h = pfsm.Handle(N, c.P, c.window, c.iters, p.alpha)
    dA = dev(p.A)
    dV = torch.empty((N, N), dtype=torch.float64, device="cuda")
    dl = torch.empty((N,), dtype=torch.float64, device="cuda")
    h.solve(dA, dV, dl)
    ref_l, ref_V, ref_e = dl.clone(), dV.clone(), h.shifts()
    for _ in range(reps):
        dV.fill_(float("nan"))
        dl.fill_(float("nan"))
        h.solve(dA, dV, dl)
        assert torch.equal(dl, ref_l) and torch.equal(dV, ref_V) and torch.equal(h.shifts(), ref_e)
    assert h.info() == 0
    h.destroy()
