"""Pins for the CPU oracle: what the paper and the mathematics fix.

The paper prints no worked numerical example, so every pin is a closed form, an invariant, a special
case that reduces to a library routine (numpy.linalg.eigh / qr / cholesky are used ONLY here, as an
independent check -- the oracle itself contains no library linear algebra), or brute force on tiny
inputs.  Each test says which plausible mistake it would catch.
"""
import os

import numpy as np
import pytest

import oracle
import pfsm_inputs as gen

pytestmark = pytest.mark.filterwarnings("ignore")


def known_spectrum_matrix(N, d, seed, nreflect=3):
    Q = gen.householder_orthogonal(N, nreflect, seed)
    A = (Q * d) @ Q.T
    return 0.5 * (A + A.T), Q


# ---------------------------------------------------------------- O1 partition (R6/R7)
def test_partition_hand_case():
    # N=12, P=3, w=1: m=4, M=6.  Interior slice centred, end slices shifted inward (same M everywhere).
    M, g0, lo, off = oracle.partition(12, 3, 1)
    assert M == 6
    assert g0.tolist() == [0, 4, 8]
    assert lo.tolist() == [0, 3, 6]      # clamp(g0 - w, 0, N - M)
    assert off.tolist() == [0, 1, 2]     # local index of the slice's first eigenpair


def test_partition_baseline_configs():
    for c in gen.CONFIGS:
        M, g0, lo, off = oracle.partition(c.N, c.P, c.window)
        assert M == c.m + 2 * c.window == c.M
        assert np.all(lo >= 0) and np.all(lo + M <= c.N)
        assert np.all(off >= 0) and np.all(off + c.m <= M)
        assert off[0] == 0 and off[-1] == M - c.m
        if c.P > 2:
            assert np.all(off[1:-1] == c.window)


def test_partition_wide_window_and_bad_args():
    M, g0, lo, off = oracle.partition(16, 4, 100)
    assert M == 16 and lo.tolist() == [0, 0, 0, 0] and off.tolist() == [0, 4, 8, 12]
    for bad in [(10, 0, 1), (10, 11, 1), (10, 3, -1), (0, 1, 0)]:
        with pytest.raises(ValueError):
            oracle.partition(*bad)


def test_partition_uneven_hand_case():
    # R14: N = 10, P = 3, w = 1.  g0 = floor(s N / P) = 0, 3, 6: slices of 3, 3 and 4 eigenpairs; every
    # submatrix has order ceil(10/3) + 2 = 6; lo = clamp(g0 - 1, 0, 4), off = g0 - lo.
    M, g0, lo, off = oracle.partition(10, 3, 1)
    assert M == 6
    assert g0.tolist() == [0, 3, 6] and oracle.slice_counts(10, 3).tolist() == [3, 3, 4]
    assert lo.tolist() == [0, 2, 4] and off.tolist() == [0, 1, 2]


@pytest.mark.parametrize("N,P,w", [(10, 3, 1), (250, 7, 9), (97, 5, 0), (1664, 12, 100), (64, 64, 2), (50, 49, 3), (31, 4, 40)])
def test_partition_invariants_any_sizes(N, P, w):
    M, g0, lo, off = oracle.partition(N, P, w)
    cnt = oracle.slice_counts(N, P)
    assert cnt.sum() == N and cnt.min() >= N // P and cnt.max() <= -(-N // P)      # slices tile 0..N-1, sizes differ by <= 1
    assert np.array_equal(g0, np.concatenate([[0], np.cumsum(cnt)[:-1]]))
    assert M == min(N, cnt.max() + 2 * w)
    assert np.all(lo >= 0) and np.all(lo + M <= N)                                 # window inside the matrix
    assert np.all(off == g0 - lo) and np.all(off >= 0) and np.all(off + cnt <= M)  # the slice's rows are inside its window
    inner = (g0 - w >= 0) & (g0 - w + M <= N)
    assert np.all(off[inner] == w)                                                 # unclamped windows are centred (halo w below)
    if N % P == 0:
        assert np.all(cnt == N // P)


# ---------------------------------------------------------------- P6: 2x2 / 3x3 hand cases
def test_jacobi_2x2_closed_form():
    a, b, c = 2.0, -0.75, -1.0
    mu, Y, sw = oracle.jacobi_eig(np.array([[a, b], [b, c]]))
    mid, rad = 0.5 * (a + c), np.hypot(0.5 * (a - c), b)
    np.testing.assert_allclose(mu, [mid - rad, mid + rad], rtol=0, atol=1e-15)
    B = np.array([[a, b], [b, c]])
    np.testing.assert_allclose(B @ Y, Y * mu, atol=1e-15)
    assert sw >= 1


def test_jacobi_3x3_hand_case():
    # [[2,1,0],[1,2,1],[0,1,2]] has eigenvalues 2 - sqrt2, 2, 2 + sqrt2 (tridiagonal Toeplitz closed form)
    B = np.array([[2.0, 1, 0], [1, 2, 1], [0, 1, 2]])
    mu, Y, _ = oracle.jacobi_eig(B)
    np.testing.assert_allclose(mu, [2 - np.sqrt(2), 2, 2 + np.sqrt(2)], atol=2e-15)
    v = np.abs(Y[:, 1])
    np.testing.assert_allclose(v, [np.sqrt(0.5), 0, np.sqrt(0.5)], atol=1e-15)


def test_jacobi_sort_is_ascending_and_stable_on_ties():
    mu, Y, _ = oracle.jacobi_eig(np.diag([3.0, 1.0, 3.0, -2.0]))
    assert mu.tolist() == [-2.0, 1.0, 3.0, 3.0]
    # ties keep the lower original index first: e_0 before e_2
    assert np.argmax(np.abs(Y[:, 2])) == 0 and np.argmax(np.abs(Y[:, 3])) == 2


# ---------------------------------------------------------------- P4: known spectrum Q diag(d) Q^T
@pytest.mark.parametrize("N", [5, 32, 97])
def test_jacobi_known_spectrum(N):
    d = np.sort(gen.uniform(11, gen.STREAM_TEST, 10_000, N) * 4 - 2)
    A, Q = known_spectrum_matrix(N, d, seed=12 + N)
    mu, Y, sw = oracle.jacobi_eig(A)
    nA = np.linalg.norm(A)
    assert sw > 0
    np.testing.assert_allclose(mu, d, atol=1e-14 * nA)
    assert np.abs(Y.T @ Y - np.eye(N)).max() < 1e-14 * N
    assert np.abs(A @ Y - Y * mu).max() < 1e-14 * nA
    # and against the library routine
    np.testing.assert_allclose(mu, np.linalg.eigvalsh(A), atol=1e-14 * nA)


# ---------------------------------------------------------------- P1: diagonal A is a fixed point of every step
@pytest.mark.parametrize("P,w,iters", [(4, 3, 2), (1, 0, 1), (8, 0, 3), (2, 100, 4), (5, 2, 2), (7, 0, 1), (31, 1, 2)])
def test_diagonal_input_exact(P, w, iters):
    N = 32
    d = np.sort(gen.uniform(5, gen.STREAM_TEST, 0, N) * 2 - 1)
    r = oracle.pfsm(np.diag(d), P, w, iters, 0.5)
    assert r["info"] == 0
    assert np.array_equal(r["lam"], d)          # bitwise
    assert np.array_equal(r["eps"], d)
    assert np.array_equal(r["Vr"], np.eye(N))
    assert np.array_equal(r["resid"], np.zeros(N))


def test_diagonal_input_with_exact_degeneracy():
    N = 24
    d = np.repeat(np.arange(6.0), 4)  # 4-fold degenerate levels: only invariants are checked (R16)
    r = oracle.pfsm(np.diag(d), 4, 2, 2, 0.01)
    assert r["info"] == 0
    np.testing.assert_allclose(np.sort(r["lam"]), d, atol=1e-15)
    assert np.abs(r["Vr"] @ r["Vr"].T - np.eye(N)).max() < 1e-15
    assert r["resid"].max() < 1e-15


# ---------------------------------------------------------------- P2: slice-aligned block-diagonal A
@pytest.mark.parametrize("w", [0, 2, 5])
def test_block_diagonal_slices_exact(w):
    # blocks = slices, block s has spectrum inside [10 s, 10 s + 1]: by Cauchy interlacing the halo adds
    # exactly `off` eigenvalues below the slice's range, so local indices off..off+m-1 (R7) are exactly
    # block s's eigenpairs, incl. the clamped end slices (R6).  A wrong lo/off rule fails here.
    P, m = 4, 6
    N = P * m
    A = np.zeros((N, N))
    expected = []
    for s in range(P):
        d = 10.0 * s + np.sort(gen.uniform(77, gen.STREAM_TEST, 100 * s, m))
        Bs, _ = known_spectrum_matrix(m, d, seed=300 + s, nreflect=2)
        A[s * m:(s + 1) * m, s * m:(s + 1) * m] = Bs
        expected.append(np.linalg.eigvalsh(Bs))
    expected = np.concatenate(expected)
    r = oracle.pfsm(A, P, w, 2, 0.5 / 31.0 ** 2)
    assert r["info"] == 0
    nA = np.linalg.norm(A)
    np.testing.assert_allclose(r["lam"], expected, atol=1e-14 * nA)   # in slice order, not re-sorted (R12)
    np.testing.assert_allclose(r["eps"], expected, atol=1e-14 * nA)   # shifts are the submatrix eigenvalues (R8)
    assert r["resid"].max() < 1e-14 * nA
    # start vectors are zero outside their own block
    V = r["Vr"]
    for s in range(P):
        rows = V[s * m:(s + 1) * m]
        mask = np.ones(N, bool)
        mask[s * m:(s + 1) * m] = False
        assert np.abs(rows[:, mask]).max() < 1e-15


@pytest.mark.parametrize("w", [0, 3])
def test_block_diagonal_uneven_slices_exact(w):
    # Same pin with P not dividing N (R14): N = 22, P = 4 -> slices of 5, 6, 5, 6 eigenpairs at g0 = 0, 5, 11, 16.
    # Blocks = slices, spectra separated, so slice s must return exactly block s's eigenpairs; a wrong slice size,
    # start or window offset mixes neighbouring blocks and fails.
    N, P = 22, 4
    cnt = oracle.slice_counts(N, P)
    assert cnt.tolist() == [5, 6, 5, 6]
    g0 = np.concatenate([[0], np.cumsum(cnt)])
    A = np.zeros((N, N))
    expected = []
    for s in range(P):
        d = 10.0 * s + np.sort(gen.uniform(78, gen.STREAM_TEST, 100 * s, int(cnt[s])))
        Bs, _ = known_spectrum_matrix(int(cnt[s]), d, seed=400 + s, nreflect=2)
        A[g0[s]:g0[s + 1], g0[s]:g0[s + 1]] = Bs
        expected.append(np.linalg.eigvalsh(Bs))
    expected = np.concatenate(expected)
    r = oracle.pfsm(A, P, w, 2, 0.5 / 31.0 ** 2)
    assert r["info"] == 0
    nA = np.linalg.norm(A)
    np.testing.assert_allclose(r["lam"], expected, atol=1e-14 * nA)
    np.testing.assert_allclose(r["eps"], expected, atol=1e-14 * nA)
    assert r["resid"].max() < 1e-14 * nA
    V = r["Vr"]
    for s in range(P):
        mask = np.ones(N, bool)
        mask[g0[s]:g0[s + 1]] = False
        assert np.abs(V[g0[s]:g0[s + 1]][:, mask]).max() < 1e-15


# ---------------------------------------------------------------- P3: P=1 or m+2w >= N reduces to a full eigensolve
@pytest.mark.parametrize("P,w", [(1, 0), (4, 40), (3, 40), (7, 20)])
def test_full_window_reduces_to_eigh(P, w):
    N = 40
    p = gen.small_problem(N, 0.05, 6.0, seed=9)
    r = oracle.pfsm(p.A, P, w, 3, p.alpha)
    ex = np.linalg.eigvalsh(p.A)
    nA = np.linalg.norm(p.A)
    assert r["info"] == 0
    np.testing.assert_allclose(r["lam"], ex, atol=1e-14 * nA)
    assert r["resid"].max() < 1e-13 * nA
    assert np.abs(r["Vr"] @ r["Vr"].T - np.eye(N)).max() < 1e-13


# ---------------------------------------------------------------- step 2 start vectors
@pytest.mark.parametrize("N,P,w", [(48, 4, 5), (50, 4, 5), (47 + 1, 7, 3)])
def test_step2_zero_padding_and_shifts(N, P, w):
    p = gen.small_problem(N, 0.02, 4.0, seed=21)
    M, g0, lo, off = oracle.partition(N, P, w)
    Vr, eps, info = oracle.step2(p.A, P, w)
    assert info == 0
    cnt = oracle.slice_counts(N, P)
    for s in range(P):
        B = p.A[lo[s]:lo[s] + M, lo[s]:lo[s] + M]
        mu, Y = np.linalg.eigh(B)
        for j in range(cnt[s]):
            i = g0[s] + j
            assert abs(eps[i] - mu[off[s] + j]) < 1e-14
            v = Vr[i]
            outside = np.ones(N, bool)
            outside[lo[s]:lo[s] + M] = False
            assert np.all(v[outside] == 0.0)                     # exactly zero
            y = Y[:, off[s] + j]
            inside = v[lo[s]:lo[s] + M]
            assert min(np.abs(inside - y).max(), np.abs(inside + y).max()) < 1e-12   # sign freedom (R16)
            assert abs(np.linalg.norm(inside) - 1) < 1e-14


# ---------------------------------------------------------------- P5: closed-form iterate of Eq. 6-7
@pytest.mark.parametrize("iters", [1, 2, 5])
def test_step3_closed_form_factor(iters):
    # A = Q diag(d) Q^T, any start x, fixed shift eps:
    #   x_j = Q diag((1 - alpha (d_k - eps)^2)^j) Q^T x_0
    # A linear (one-product) reading of step 3, a wrong sign of alpha, a shift applied once, or a
    # normalization between iterations all fail this.
    N = 24
    d = np.sort(gen.uniform(3, gen.STREAM_TEST, 0, N) * 3 - 1)
    A, Q = known_spectrum_matrix(N, d, seed=4)
    X0 = gen.normal(8, gen.STREAM_TEST, 0, N * N).reshape(N, N)   # row i = x_i^0
    eps = gen.uniform(8, gen.STREAM_TEST, 5000, N) * 3 - 1
    alpha = 0.5 / np.max(np.abs(d)) ** 2
    got = oracle.step3(A, X0, eps, iters, alpha)
    for i in range(N):
        f = (1.0 - alpha * (d - eps[i]) ** 2) ** iters
        want = Q @ (f * (Q.T @ X0[i]))
        np.testing.assert_allclose(got[i], want, atol=1e-13)


def test_step3_column_range_only_touches_requested_columns():
    N = 16
    p = gen.small_problem(N, 0.05, 3.0, seed=2)
    X0 = gen.normal(9, gen.STREAM_TEST, 0, N * N).reshape(N, N)
    eps = np.zeros(N)
    full = oracle.step3(p.A, X0, eps, 2, p.alpha)
    part = oracle.step3(p.A, X0, eps, 2, p.alpha, 3, 9)
    assert np.array_equal(part[3:9], full[3:9])
    assert np.array_equal(part[:3], X0[:3]) and np.array_equal(part[9:], X0[9:])


# ---------------------------------------------------------------- step 4: Gram-Schmidt == thin QR with positive diagonal R
def test_step4_matches_qr_uniqueness():
    N = 30
    X = gen.normal(17, gen.STREAM_TEST, 0, N * N).reshape(N, N) + 3 * np.eye(N)
    Vr, info = oracle.step4_mgs(X)
    assert info == 0
    Qn, Rn = np.linalg.qr(X.T)            # columns of X.T are the vectors
    Qn = Qn * np.sign(np.diag(Rn))        # make diag(R) positive -> unique factor
    np.testing.assert_allclose(Vr.T, Qn, atol=1e-13)
    # V_out^T V_in = R must be upper triangular with positive diagonal (ascending column order, R10)
    R = Vr @ X.T
    assert np.abs(np.tril(R, -1)).max() < 1e-13
    assert np.all(np.diag(R) > 0)


def test_step4_breakdown_flag():
    # P12: duplicate column -> breakdown reported at the second copy (1-based)
    N = 12
    X = gen.normal(18, gen.STREAM_TEST, 0, N * N).reshape(N, N)
    X[7] = X[2]
    _, info = oracle.step4_mgs(X)
    assert info == 8


# ---------------------------------------------------------------- step 5 against the definition
def test_step5_definition():
    N = 20
    p = gen.small_problem(N, 0.1, 3.0, seed=33)
    X = gen.normal(19, gen.STREAM_TEST, 0, N * N).reshape(N, N)
    X /= np.linalg.norm(X, axis=1, keepdims=True)
    lam, res = oracle.step5(p.A, X)
    for i in range(N):
        t = p.A @ X[i]
        li = X[i] @ t
        assert abs(lam[i] - li) < 1e-14
        assert abs(res[i] - np.linalg.norm(t - li * X[i])) < 1e-14


# ---------------------------------------------------------------- P7, P8, P9 on a config-0-shaped problem
@pytest.fixture(scope="module")
def cfg0():
    p = gen.problem(0)
    c = p.cfg
    return p, oracle.pfsm(p.A, c.P, c.window, c.iters, p.alpha)


def test_config0_invariants(cfg0):
    p, r = cfg0
    N = p.cfg.N
    V = r["Vr"]
    assert r["info"] == 0
    assert abs(r["lam"].sum() - np.trace(p.A)) < 1e-12 * N                    # P7 trace
    assert np.abs(V @ V.T - np.eye(N)).max() < 1e-12 * N                      # P8 orthonormality
    ex = np.linalg.eigvalsh(p.A)
    dist = np.abs(r["lam"][:, None] - ex[None, :]).min(axis=1)
    assert np.all(dist <= r["resid"] + 1e-13)                                # P9 residual enclosure
    # step 5 is consistent with the returned vectors
    t = V @ p.A
    np.testing.assert_allclose(r["lam"], np.einsum("ij,ij->i", V, t), atol=1e-13)
    # PFSM is an approximation here (narrow window): information, matches SURVEY.md's pre-check scale
    assert 1e-7 < np.abs(np.sort(r["lam"]) - ex).max() < 1e-4


def test_config0_golden_summary(cfg0):
    # tests/golden/config0_oracle.txt is written by tests/golden/make_golden.py, which calls only oracle/
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "config0_oracle.txt")
    vals = {}
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()
        vals[k] = float(v)
    p, r = cfg0
    assert abs(r["lam"].sum() - vals["sum_lambda"]) < 1e-11
    assert abs(r["lam"][0] - vals["lambda_0"]) < 1e-12
    assert abs(r["lam"][-1] - vals["lambda_255"]) < 1e-12
    assert abs(r["resid"].max() - vals["max_resid"]) < 1e-12


# ---------------------------------------------------------------- P10: brute force vs full Jacobi at N <= 64
def test_bruteforce_small_wide_window():
    N, P, w = 64, 4, 12     # M = 40 = 0.625 N (paper recommends >= 0.3 N)
    p = gen.small_problem(N, 2e-3, 8.0, seed=41)
    mu, Y, _ = oracle.jacobi_eig(p.A)       # O6: exact spectrum
    errs = []
    for iters in (0, 2, 6):
        r = oracle.pfsm(p.A, P, w, iters, p.alpha)
        assert r["info"] == 0
        dist = np.abs(r["lam"][:, None] - mu[None, :]).min(axis=1)
        assert np.all(dist <= r["resid"] + 1e-13)        # P9
        assert abs(r["lam"].sum() - np.trace(p.A)) < 1e-12
        errs.append(np.abs(np.sort(r["lam"]) - mu).max())
        # second-order accuracy of Rayleigh quotients: |lambda - exact| <= r^2 / gap-ish; crude bound r
        assert errs[-1] <= r["resid"].max()
    assert errs[0] < 1e-5


def test_iters0_is_gram_schmidt_of_start_vectors():
    # with iters = 0 the result is O2 + O4 + O5 only
    N, P, w = 48, 4, 4
    p = gen.small_problem(N, 0.01, 5.0, seed=43)
    r = oracle.pfsm(p.A, P, w, 0, p.alpha)
    V0, eps, _ = oracle.step2(p.A, P, w)
    Vg, info = oracle.step4_mgs(V0)
    lam, res = oracle.step5(p.A, Vg)
    assert np.array_equal(r["Vr"], Vg) and np.array_equal(r["lam"], lam) and np.array_equal(r["resid"], res)


def test_iterations_reduce_residuals():
    # folded-spectrum iterations must pull each vector toward the eigenvector nearest its shift
    N, P, w = 96, 4, 6
    p = gen.small_problem(N, 5e-3, 8.0, seed=47)
    r0 = oracle.pfsm(p.A, P, w, 0, p.alpha)
    r8 = oracle.pfsm(p.A, P, w, 8, p.alpha)
    assert r8["resid"].max() < r0["resid"].max()
    assert np.median(r8["resid"]) < np.median(r0["resid"])


# ---------------------------------------------------------------- P12: the paper's failure mode
def test_randomly_mixed_eigenvectors_degrade():
    # A = Q D Q^T with a dense random Q is not diagonally dominant: submatrix eigenvectors mix the whole
    # spectrum, the method "will not work reliably".  Either breakdown is flagged or the residuals are huge.
    N, P, w = 48, 4, 4
    d = np.sort(gen.uniform(51, gen.STREAM_TEST, 0, N) * 2 - 1)
    X = gen.normal(51, gen.STREAM_TEST, 10_000, N * N).reshape(N, N)
    Q, _ = np.linalg.qr(X)
    A = (Q * d) @ Q.T
    A = 0.5 * (A + A.T)
    r = oracle.pfsm(A, P, w, 3, 0.5)
    good = gen.small_problem(N, 1e-3, 8.0, seed=51)
    rg = oracle.pfsm(good.A, P, w, 3, good.alpha)
    assert r["info"] != 0 or r["resid"].max() > 100 * rg["resid"].max()


# ---------------------------------------------------------------- P13: generalized variant
def test_generalized_identity_overlap_is_a_no_op():
    N = 24
    p = gen.small_problem(N, 0.01, 4.0, seed=61)
    L, Ap, info = oracle.generalized_reduce(p.A, np.eye(N))
    assert info == 0
    assert np.array_equal(L, np.eye(N)) and np.array_equal(Ap, p.A)
    X = gen.normal(61, gen.STREAM_TEST, 0, N * N).reshape(N, N)
    assert np.array_equal(oracle.generalized_back(L, X), X)


def test_generalized_against_library():
    N, P, w = 40, 4, 40   # full window -> exact
    p = gen.small_problem(N, 0.01, 4.0, seed=62)
    S = gen.banded_symmetric(N, np.ones(N), 1e-2, 6.0, 62, gen.STREAM_S)
    L, Ap, info = oracle.generalized_reduce(p.A, S)
    assert info == 0
    np.testing.assert_allclose(L, np.linalg.cholesky(S), atol=1e-14)
    Li = np.linalg.inv(np.linalg.cholesky(S))
    np.testing.assert_allclose(Ap, Li @ p.A @ Li.T, atol=1e-13)
    r = oracle.pfsm(Ap, P, w, 2, p.alpha)
    Xr = oracle.generalized_back(L, r["Vr"])
    assert np.abs(Xr @ S @ Xr.T - np.eye(N)).max() < 1e-12 * N           # X^T S X = I
    resid = Xr @ p.A - (Xr @ S) * r["lam"][:, None]
    assert np.abs(resid).max() < 1e-12
    import scipy.linalg
    np.testing.assert_allclose(r["lam"], scipy.linalg.eigh(p.A, S, eigvals_only=True), atol=1e-12)


def test_generalized_reduce_flags_indefinite_overlap():
    S = np.eye(4)
    S[2, 2] = -1.0
    _, _, info = oracle.generalized_reduce(np.eye(4), S)
    assert info == 3


# ---------------------------------------------------------------- SCF-sequence mode
def test_warm_start_identity_basis_is_plain_pfsm():
    N, P, w = 48, 4, 5
    p = gen.small_problem(N, 0.01, 5.0, seed=81)
    a = oracle.pfsm(p.A, P, w, 2, p.alpha)
    b = oracle.pfsm_warm(p.A, np.eye(N), P, w, 2, p.alpha)
    assert np.array_equal(a["lam"], b["lam"]) and np.array_equal(a["Vr"], b["Vr"])


def test_warm_start_with_exact_previous_eigenvectors_is_exact():
    # V_prev = eigenvectors of A itself -> A' is diagonal -> fixed point of every step (P1), for ANY dense A:
    # this is the paper's point that a good previous solution makes the method applicable.
    N, P, w = 40, 4, 3
    d = np.sort(gen.uniform(82, gen.STREAM_TEST, 0, N) * 2 - 1)
    X = gen.normal(82, gen.STREAM_TEST, 10_000, N * N).reshape(N, N)
    Q, _ = np.linalg.qr(X)
    A = (Q * d) @ Q.T
    A = 0.5 * (A + A.T)
    lam0, V0 = np.linalg.eigh(A)
    r = oracle.pfsm_warm(A, V0.T.copy(), P, w, 2, 0.5)
    assert r["info"] == 0
    np.testing.assert_allclose(r["lam"], lam0, atol=1e-13)
    assert np.abs(r["Vr"] @ r["Vr"].T - np.eye(N)).max() < 1e-13
    assert np.abs(r["Vr"] @ A - r["lam"][:, None] * r["Vr"]).max() < 1e-13


def test_warm_start_tracks_a_slowly_changing_matrix():
    # a sequence A_k = A_0 + k dA with dense small dA: each step starts from the previous step's vectors
    N, P, w = 64, 4, 8
    d = np.sort(gen.uniform(83, gen.STREAM_TEST, 0, N) * 2 - 1)
    X = gen.normal(83, gen.STREAM_TEST, 10_000, N * N).reshape(N, N)
    Q, _ = np.linalg.qr(X)
    A0 = (Q * d) @ Q.T
    dA = gen.normal(83, gen.STREAM_TEST, 50_000, N * N).reshape(N, N) * 2e-4
    dA = 0.5 * (dA + dA.T)
    _, V = np.linalg.eigh(0.5 * (A0 + A0.T))
    Vr = V.T.copy()
    for k in range(1, 4):
        Ak = 0.5 * (A0 + A0.T) + k * dA
        r = oracle.pfsm_warm(Ak, Vr, P, w, 3, 0.5)
        assert r["info"] == 0
        ex = np.linalg.eigvalsh(Ak)
        assert np.abs(np.sort(r["lam"]) - ex).max() < 1e-5
        assert abs(r["lam"].sum() - np.trace(Ak)) < 1e-12          # P7 for the rotated basis too
        Vr = r["Vr"]


# ---------------------------------------------------------------- f2: Eq. 14-15
def test_eq14_identity_overlap_is_a_fixed_point():
    N = 20
    p = gen.small_problem(N, 0.1, 4.0, seed=91)
    for niter in (0, 1, 4):
        assert np.array_equal(oracle.eq14_iteration(p.A, np.eye(N), niter), p.A)


def test_eq14_diagonal_overlap_converges_in_one_step():
    # B = D diagonal: Z_1 = A - D^-1 (D A - A) = D^-1 A exactly (up to rounding), and stays there
    N = 16
    p = gen.small_problem(N, 0.1, 4.0, seed=92)
    dd = 1.0 + gen.uniform(92, gen.STREAM_TEST, 0, N)
    want = p.A / dd[:, None]
    np.testing.assert_allclose(oracle.eq14_iteration(p.A, np.diag(dd), 1), want, atol=1e-15)
    np.testing.assert_allclose(oracle.eq14_iteration(p.A, np.diag(dd), 3), want, atol=1e-15)


def test_eq14_error_contracts_with_the_jacobi_iteration_matrix():
    # Z_n - B^-1 A = (I - D^-1 B)^n (Z_0 - B^-1 A): closed form of the stationary iteration (Eq. 15 at the
    # fixed point gives B Z = A).  A sign error, D^-1 on the wrong side, or Z_0 = I all fail this.
    N = 24
    p = gen.small_problem(N, 0.1, 4.0, seed=93)
    B = gen.banded_symmetric(N, np.ones(N), 2e-2, 5.0, 93, gen.STREAM_S)
    exact = np.linalg.solve(B, p.A)
    Mj = np.eye(N) - B / np.diag(B)[:, None]
    for n in (1, 2, 5):
        want = exact + np.linalg.matrix_power(Mj, n) @ (p.A - exact)
        np.testing.assert_allclose(oracle.eq14_iteration(p.A, B, n), want, atol=1e-14)
    Z = oracle.eq14_iteration(p.A, B, 40)
    assert np.abs(B @ Z - p.A).max() < 1e-14
    Zs = oracle.eq14_iteration(p.A, B, 40, symmetrize=True)
    assert np.array_equal(Zs, Zs.T)


# ---------------------------------------------------------------- seeded sweep of shapes: invariants that hold for ANY PFSM run
def _oracle_sweep_cases(count=14):
    u = gen.uniform(424242, gen.STREAM_TEST, 0, 4 * count)
    out = []
    for k in range(count):
        N = 2 * int(3 + u[4 * k] * 45)                       # 6 .. 94
        divs = [d for d in range(1, N + 1) if N % d == 0]
        P = divs[int(u[4 * k + 1] * len(divs)) % len(divs)]
        if k % 3 == 2:
            P = 1 + int(u[4 * k + 1] * min(N, 12))               # any P: uneven slices (R14)
        out.append((N, P, int(u[4 * k + 2] * 12), int(u[4 * k + 3] * 5)))
    return out


@pytest.mark.parametrize("N,P,w,iters", _oracle_sweep_cases())
def test_oracle_invariants_on_a_seeded_sweep(N, P, w, iters):
    p = gen.small_problem(N, 2e-3, max(2.0, N / 8.0), seed=7000 + N + P)
    r = oracle.pfsm(p.A, P, w, iters, p.alpha)
    assert r["info"] == 0
    V = r["Vr"]
    assert np.abs(V @ V.T - np.eye(N)).max() < 1e-12 * N                       # P8
    assert abs(r["lam"].sum() - np.trace(p.A)) < 1e-12 * N                    # P7
    ex = np.linalg.eigvalsh(p.A)
    assert np.all(np.abs(r["lam"][:, None] - ex[None, :]).min(axis=1) <= r["resid"] + 1e-13)   # P9
    np.testing.assert_allclose(r["lam"], np.einsum("ij,ij->i", V @ p.A, V), atol=1e-13)         # step 5 definition
    # slice structure: the shifts of slice s are m consecutive eigenvalues of its own submatrix (R7)
    M, g0, lo, off = oracle.partition(N, P, w)
    cnt = oracle.slice_counts(N, P)
    for s in range(P):
        mu = np.linalg.eigvalsh(p.A[lo[s]:lo[s] + M, lo[s]:lo[s] + M])
        np.testing.assert_allclose(r["eps"][g0[s]:g0[s] + cnt[s]], mu[off[s]:off[s] + cnt[s]], atol=1e-13)


@pytest.mark.parametrize("k", [3, 4])
def test_large_golden_files_belong_to_the_generators_matrix(k):
    """tests/golden/config{3,4}_oracle.txt hold the oracle's full output for the two configs whose oracle run takes
    minutes.  They must describe the matrix pfsm_inputs builds today (alpha, ||A||_F) and satisfy what holds for any
    orthonormal V: sum(lambda) = trace(A) (pin P7), ||V^T V - I||_max within the gate, r >= 0, N rows."""
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", f"config{k}_oracle.txt")
    head, rows = {}, []
    for ln in open(path):
        if ln.startswith("#"):
            continue
        f = ln.split()
        if len(f) == 2:
            head[f[0]] = float(f[1])
        elif len(f) == 3:
            rows.append([float(x) for x in f])
    arr = np.array(rows)
    c = gen.config(k)
    d = gen.spectrum(k)
    assert int(head["N"]) == c.N and arr.shape == (c.N, 3)
    assert head["alpha"] == gen.alpha_rule(d)
    A = gen.banded_symmetric(c.N, d, c.amp, c.width, c.seed, gen.STREAM_E)
    nF = float(np.sqrt(np.sum(A * A)))
    assert abs(head["normF"] - nF) <= 1e-12 * nF
    assert abs(arr[:, 0].sum() - np.trace(A)) <= 1e-9            # P7: trace invariant
    assert head["ortho_max"] <= 1e-12 * c.N
    assert np.all(arr[:, 1] >= 0.0)
    # shifts are eigenvalues of principal submatrices: inside A's Gershgorin range; lambda are Rayleigh quotients: same
    gl = (np.diag(A) - (np.abs(A).sum(1) - np.abs(np.diag(A)))).min()
    gh = (np.diag(A) + (np.abs(A).sum(1) - np.abs(np.diag(A)))).max()
    assert arr[:, 0].min() >= gl and arr[:, 0].max() <= gh and arr[:, 2].min() >= gl and arr[:, 2].max() <= gh
    vec = np.load(path.replace(".txt", "_vectors.npz"))
    assert np.abs(np.einsum("ij,ij->i", vec["Vr"], vec["Vr"]) - 1.0).max() < 1e-13
    lam_chk = np.einsum("ij,ij->i", vec["Vr"] @ A, vec["Vr"])       # Rayleigh quotients of the stored vectors
    assert np.abs(lam_chk - arr[vec["idx"], 0]).max() <= 1e-12 * nF
