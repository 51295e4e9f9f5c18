/*
 * pfsm_oracle.cpp -- CPU oracle for one partitioned-folded-spectrum (PFSM) solve.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code with the
 * CUDA path under paper_1502_07806_b200/csrc (no headers, helpers, tables or constants).
 *
 * Plain, slow, FP64, column-major (ld = N), OpenMP over independent columns only.  Every
 * function follows the paper (arXiv 1502.07806, /root/reference/PAPER.md) in its order and
 * notation; readings R1..R20 of SURVEY.md §8(c) (restated in DESIGN.md) fill the gaps.
 *
 *   O1 oracle_partition      PAPER.md:88  (§II: "slice of eigenvectors of size m = N/P",
 *                                          "each diagonal submatrix B is of order M")
 *   O2 oracle_jacobi_eig     PAPER.md:86-94 (§II: "B y_i = lambda y_i"); textbook cyclic Jacobi
 *      oracle_step2          PAPER.md:94  (start vectors x_i^0 zero-padded, shifts = eigenvalues)
 *   O3 oracle_step3          PAPER.md:83  (Eq. 11: x <- x - alpha (A - eps I)^2 x, applied as two
 *                                          successive products)
 *   O4 oracle_step4_mgs      PAPER.md:94-96 ("Gram-Schmidt orthogonalization")
 *   O5 oracle_step5          north_star step 5 (paper silent, reading R11): Rayleigh quotients
 *   OG oracle_generalized_*  BASELINE.json configs[4] / PAPER.md:171-173 (Eq. 13)
 *   f2 oracle_eq14_iteration PAPER.md:173-185 (Eq. 14-15: Z = B^-1 A by a column-parallel iteration)
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): P1 diagonal input, P2 slice-aligned block
 * diagonal, P3 P=1 / window >= N vs numpy eigh, P4 known spectrum Q diag(d) Q^T, P5 closed-form
 * iterate of Eq. 6-7, P6 2x2/3x3 hand cases, P7 trace, P8 orthonormality, P9 residual enclosure,
 * P10 brute force at N <= 64, P12 negative test, P13 generalized variant.
 * Parity unpinned: the accuracy of PFSM relative to the exact spectrum at configs 1-4 (the paper
 * prints no tolerances; Figs. 2-4 are images) -- reported as information only.
 */
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <numeric>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {

/* ---------------------------------------------------------------------------------------------
 * O1  Partition (readings R6, R7, R14).
 * Slice s holds the eigen-indices g0[s] .. g0[s+1]-1 with g0[s] = floor(s N / P) (m = N/P of them when P divides N,
 * the paper's case; otherwise floor(N/P) or ceil(N/P) -- R14).  Every submatrix has the same order
 * M = min(N, ceil(N/P) + 2w); lo = clamp(g0 - w, 0, N - M), off = g0 - lo.
 * g0 has P + 1 entries (g0[P] = N).  Returns M, or -1 for bad sizes (P > N leaves a slice empty).
 * ------------------------------------------------------------------------------------------- */
int64_t oracle_partition(int64_t N, int64_t P, int64_t w, int64_t* g0, int64_t* lo, int64_t* off) {
    if (N < 1 || P < 1 || w < 0 || P > N) return -1;
    const int64_t mmax = (N + P - 1) / P;
    const int64_t M = std::min<int64_t>(N, mmax + 2 * w);
    for (int64_t s = 0; s < P; ++s) {
        g0[s] = (s * N) / P;
        lo[s] = std::min<int64_t>(std::max<int64_t>(g0[s] - w, 0), N - M);
        off[s] = g0[s] - lo[s];
    }
    g0[P] = N;
    return M;
}

/* ---------------------------------------------------------------------------------------------
 * O2  Cyclic two-sided Jacobi eigensolver for a real symmetric n x n matrix (textbook:
 * Golub & Van Loan "Matrix Computations" §8.5, row-cyclic order).
 *   B   : n x n column-major, symmetric; destroyed.
 *   mu  : n eigenvalues, ascending (stable sort: ties keep the lower original index).
 *   Y   : n x n column-major, column k = eigenvector of mu[k].
 * Rotates until max_{p!=q} |B_pq| <= 1e-15 * ||B||_F, at most 30 sweeps.
 * Returns the number of sweeps used, or -1 if the cap was hit.
 * ------------------------------------------------------------------------------------------- */
int oracle_jacobi_eig(int64_t n, double* B, double* mu, double* Y) {
    std::vector<double> Q((size_t)n * n, 0.0);
    for (int64_t i = 0; i < n; ++i) Q[i + i * n] = 1.0;
    double fro = 0.0;
    for (int64_t k = 0; k < n * n; ++k) fro += B[k] * B[k];
    fro = std::sqrt(fro);
    const double tol = 1e-15 * fro;
    int sweeps = 0;
    bool converged = false;
    for (; sweeps <= 30; ++sweeps) {
        double offmax = 0.0;
        for (int64_t q = 0; q < n; ++q)
            for (int64_t p = 0; p < q; ++p) offmax = std::max(offmax, std::fabs(B[p + q * n]));
        if (offmax <= tol) { converged = true; break; }
        if (sweeps == 30) break;
        for (int64_t p = 0; p < n - 1; ++p) {
            for (int64_t q = p + 1; q < n; ++q) {
                const double bpq = B[p + q * n];
                if (bpq == 0.0) continue;
                const double bpp = B[p + p * n], bqq = B[q + q * n];
                /* tan of the rotation angle, the smaller root: theta = (bqq - bpp) / (2 bpq),
                   t = sign(theta) / (|theta| + sqrt(theta^2 + 1)) */
                const double theta = (bqq - bpp) / (2.0 * bpq);
                const double t = (theta >= 0.0 ? 1.0 : -1.0) / (std::fabs(theta) + std::sqrt(theta * theta + 1.0));
                const double c = 1.0 / std::sqrt(t * t + 1.0), s = t * c;
                /* B <- J^T B J with J = [[c, s], [-s, c]] in the (p, q) plane */
                for (int64_t k = 0; k < n; ++k) {  /* columns p and q */
                    const double bkp = B[k + p * n], bkq = B[k + q * n];
                    B[k + p * n] = c * bkp - s * bkq;
                    B[k + q * n] = s * bkp + c * bkq;
                }
                for (int64_t k = 0; k < n; ++k) {  /* rows p and q */
                    const double bpk = B[p + k * n], bqk = B[q + k * n];
                    B[p + k * n] = c * bpk - s * bqk;
                    B[q + k * n] = s * bpk + c * bqk;
                }
                for (int64_t k = 0; k < n; ++k) {  /* accumulate eigenvectors Q <- Q J */
                    const double qkp = Q[k + p * n], qkq = Q[k + q * n];
                    Q[k + p * n] = c * qkp - s * qkq;
                    Q[k + q * n] = s * qkp + c * qkq;
                }
            }
        }
    }
    std::vector<int64_t> order(n);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(),
                     [&](int64_t a, int64_t b) { return B[a + a * n] < B[b + b * n]; });
    for (int64_t k = 0; k < n; ++k) {
        mu[k] = B[order[k] + order[k] * n];
        std::memcpy(Y + k * n, Q.data() + order[k] * n, sizeof(double) * n);
    }
    return converged ? sweeps : -1;
}

/* ---------------------------------------------------------------------------------------------
 * O2  Step 2.  For each slice s: B_s = A[lo:lo+M, lo:lo+M]; B_s Y = Y diag(mu);
 * for j < m_s = g0[s+1] - g0[s]: eps[g0+j] = mu[off+j]; V[:, g0+j] = 0 except rows lo..lo+M-1 <- Y[:, off+j]
 * ("the elements of x_i that do not have a corresponding component in the submatrix solution
 * are set to zero").  Slices are independent (one per node in the paper).
 * Returns 0, or N + s + 1 if slice s's Jacobi did not converge.
 * ------------------------------------------------------------------------------------------- */
int64_t oracle_step2(int64_t N, int64_t P, int64_t w, const double* A, double* V, double* eps) {
    if (P < 1) return -1;
    std::vector<int64_t> g0(P + 1), lo(P), off(P);
    const int64_t M = oracle_partition(N, P, w, g0.data(), lo.data(), off.data());
    if (M < 0) return -1;
    int64_t info = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t s = 0; s < P; ++s) {
        std::vector<double> B((size_t)M * M), Y((size_t)M * M), mu(M);
        for (int64_t c = 0; c < M; ++c)
            for (int64_t r = 0; r < M; ++r) B[r + c * M] = A[(lo[s] + r) + (lo[s] + c) * N];
        const int sw = oracle_jacobi_eig(M, B.data(), mu.data(), Y.data());
        if (sw < 0) {
#pragma omp critical
            if (info == 0 || N + s + 1 < info) info = N + s + 1;
        }
        const int64_t m = g0[s + 1] - g0[s];
        for (int64_t j = 0; j < m; ++j) {
            const int64_t i = g0[s] + j;
            eps[i] = mu[off[s] + j];
            double* v = V + i * N;
            for (int64_t r = 0; r < N; ++r) v[r] = 0.0;
            for (int64_t r = 0; r < M; ++r) v[lo[s] + r] = Y[r + (off[s] + j) * M];
        }
    }
    return info;
}

/* out[:, c] = A x[:, c] - eps[c] x[:, c] for a block of nc columns: plain dot products, row r of
 * the symmetric A read as its column r (contiguous).  Several columns share one pass over A only
 * so that the oracle finishes in minutes at N ~ 9000; each entry is still the plain sum over k. */
static void shifted_product(int64_t N, const double* A, const double* x, const double* eps, int64_t nc,
                            double* out) {
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < N; ++r) {
        const double* a = A + r * N;
        for (int64_t c = 0; c < nc; ++c) {
            const double* xc = x + c * N;
            double sum = 0.0;
            for (int64_t k = 0; k < N; ++k) sum += a[k] * xc[k];
            out[r + c * N] = sum - eps[c] * xc[r];
        }
    }
}

/* ---------------------------------------------------------------------------------------------
 * O3  Step 3 (Eq. 11; readings R1, R8, R9).  `iters` times, for every column i:
 *     w = A v_i - eps_i v_i;   u = A w - eps_i w;   v_i <- v_i - alpha u.
 * Shifts stay fixed; no normalization between iterations.  Columns [c0, c1) only (all: 0, N).
 * ------------------------------------------------------------------------------------------- */
void oracle_step3(int64_t N, int64_t iters, double alpha, const double* A, double* V, const double* eps,
                  int64_t c0, int64_t c1) {
    const int64_t NB = 32;
    std::vector<double> Wb((size_t)N * NB), Ub((size_t)N * NB);
    for (int64_t b0 = c0; b0 < c1; b0 += NB) {
        const int64_t nc = std::min<int64_t>(NB, c1 - b0);
        double* Vb = V + b0 * N;
        for (int64_t it = 0; it < iters; ++it) {
            shifted_product(N, A, Vb, eps + b0, nc, Wb.data());
            shifted_product(N, A, Wb.data(), eps + b0, nc, Ub.data());
            for (int64_t c = 0; c < nc; ++c)
                for (int64_t r = 0; r < N; ++r) Vb[r + c * N] -= alpha * Ub[r + c * N];
        }
    }
}

/* ---------------------------------------------------------------------------------------------
 * O4  Step 4 (reading R10).  Modified Gram-Schmidt, ascending column order:
 *     for k = 0..N-1:  v_k <- v_k / ||v_k||;  for i > k: v_i <- v_i - (v_k^T v_i) v_k.
 * (Each v_i receives its projections sequentially in k order: textbook MGS.)
 * If ||v_k|| after projection < 1e-10 * its norm before any projection: return k+1 (breakdown,
 * the paper's failure mode for non-dominant A).  Returns 0 on success.
 * ------------------------------------------------------------------------------------------- */
int64_t oracle_step4_mgs(int64_t N, int64_t ncols, double* V) {
    std::vector<double> norm0(ncols);
    for (int64_t i = 0; i < ncols; ++i) {
        double s = 0.0;
        for (int64_t r = 0; r < N; ++r) s += V[r + i * N] * V[r + i * N];
        norm0[i] = std::sqrt(s);
    }
    for (int64_t k = 0; k < ncols; ++k) {
        double* vk = V + k * N;
        double s = 0.0;
        for (int64_t r = 0; r < N; ++r) s += vk[r] * vk[r];
        const double nrm = std::sqrt(s);
        if (!(nrm >= 1e-10 * norm0[k]) || nrm == 0.0) return k + 1;
        for (int64_t r = 0; r < N; ++r) vk[r] /= nrm;
#pragma omp parallel for schedule(static)
        for (int64_t i = k + 1; i < ncols; ++i) {
            double* vi = V + i * N;
            double dot = 0.0;
            for (int64_t r = 0; r < N; ++r) dot += vk[r] * vi[r];
            for (int64_t r = 0; r < N; ++r) vi[r] -= dot * vk[r];
        }
    }
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * O5  Step 5 (north_star step 5; readings R11, R12).  t_i = A v_i; lambda_i = v_i^T t_i;
 * r_i = ||t_i - lambda_i v_i||_2.  Column order kept (no re-sorting).  Columns [c0, c1).
 * ------------------------------------------------------------------------------------------- */
void oracle_step5(int64_t N, const double* A, const double* V, double* lambda, double* resid, int64_t c0,
                  int64_t c1) {
#pragma omp parallel for schedule(static)
    for (int64_t i = c0; i < c1; ++i) {
        const double* v = V + i * N;
        std::vector<double> t(N);
        for (int64_t r = 0; r < N; ++r) {
            const double* a = A + r * N;
            double sum = 0.0;
            for (int64_t k = 0; k < N; ++k) sum += a[k] * v[k];
            t[r] = sum;
        }
        double lam = 0.0;
        for (int64_t r = 0; r < N; ++r) lam += v[r] * t[r];
        double rr = 0.0;
        for (int64_t r = 0; r < N; ++r) {
            const double e = t[r] - lam * v[r];
            rr += e * e;
        }
        lambda[i] = lam;
        resid[i] = std::sqrt(rr);
    }
}

/* ---------------------------------------------------------------------------------------------
 * One PFSM solve, steps O1..O5.  A: N x N symmetric (both triangles), not
 * modified.  V: N x N output, column i = eigenvector i.  lambda, resid, eps: N each.
 * Returns info: 0 ok; -1 bad arguments; 1..N Gram-Schmidt breakdown at that column;
 * N+s+1 submatrix solver for slice s did not converge.
 * ------------------------------------------------------------------------------------------- */
int64_t oracle_pfsm(int64_t N, int64_t P, int64_t w, int64_t iters, double alpha, const double* A, double* V,
                    double* lambda, double* resid, double* eps) {
    int64_t info = oracle_step2(N, P, w, A, V, eps);
    if (info != 0) return info;
    oracle_step3(N, iters, alpha, A, V, eps, 0, N);
    info = oracle_step4_mgs(N, N, V);
    if (info != 0) return info;
    oracle_step5(N, A, V, lambda, resid, 0, N);
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * OG  Generalized variant A x = lambda S x (BASELINE.json configs[4]; Eq. 13):
 * S = L L^T (unblocked Cholesky); A' = L^-1 A L^-T by forward substitutions; A' symmetrized.
 * oracle_generalized_reduce: L (N x N col-major, lower, upper zeroed) and Ap out.  Returns 0 or
 * k+1 if pivot k is not positive.  oracle_generalized_back: X = L^-T V (back substitution).
 * ------------------------------------------------------------------------------------------- */
int64_t oracle_generalized_reduce(int64_t N, const double* A, const double* S, double* L, double* Ap) {
    std::memcpy(L, S, sizeof(double) * N * N);
    for (int64_t j = 0; j < N; ++j) {  /* left-looking column Cholesky */
        for (int64_t k = 0; k < j; ++k) {
            const double ljk = L[j + k * N];
            for (int64_t i = j; i < N; ++i) L[i + j * N] -= L[i + k * N] * ljk;
        }
        const double piv = L[j + j * N];
        if (!(piv > 0.0)) return j + 1;
        const double d = std::sqrt(piv);
        for (int64_t i = j; i < N; ++i) L[i + j * N] /= d;
        for (int64_t i = 0; i < j; ++i) L[i + j * N] = 0.0;
    }
    /* C = L^-1 A : solve L C = A column by column */
    std::vector<double> C((size_t)N * N);
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < N; ++c) {
        double* x = C.data() + c * N;
        for (int64_t i = 0; i < N; ++i) x[i] = A[i + c * N];
        for (int64_t i = 0; i < N; ++i) {
            x[i] /= L[i + i * N];
            for (int64_t r = i + 1; r < N; ++r) x[r] -= L[r + i * N] * x[i];
        }
    }
    /* A' = C L^-T  <=>  A'^T = L^-1 C^T : solve L Z = C^T, A' = Z^T */
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < N; ++c) {
        std::vector<double> x(N);
        for (int64_t i = 0; i < N; ++i) x[i] = C[c + i * N]; /* column c of C^T = row c of C */
        for (int64_t i = 0; i < N; ++i) {
            x[i] /= L[i + i * N];
            for (int64_t r = i + 1; r < N; ++r) x[r] -= L[r + i * N] * x[i];
        }
        for (int64_t i = 0; i < N; ++i) Ap[c + i * N] = x[i]; /* Z[:, c] -> row c of A' */
    }
    for (int64_t j = 0; j < N; ++j)
        for (int64_t i = 0; i < j; ++i) {
            const double a = 0.5 * (Ap[i + j * N] + Ap[j + i * N]);
            Ap[i + j * N] = a;
            Ap[j + i * N] = a;
        }
    return 0;
}

void oracle_generalized_back(int64_t N, const double* L, const double* V, double* X) {
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < N; ++c) {
        double* x = X + c * N;
        for (int64_t i = 0; i < N; ++i) x[i] = V[i + c * N];
        for (int64_t i = N - 1; i >= 0; --i) { /* L^T x = v */
            double s = x[i];
            for (int64_t r = i + 1; r < N; ++r) s -= L[r + i * N] * x[r];
            x[i] = s / L[i + i * N];
        }
    }
}

/* ---------------------------------------------------------------------------------------------
 * f2  The paper's generalized -> standard conversion (Eq. 14-15; reading R19:
 * Eq. 14 prints "D^-1 A x" where the matrix iteration needs D^-1 A).  D = diag(B);
 *     Z_0 = A   ("the identity serves as a good initial approximation" of B^-1)
 *     Z_{n+1} = (I - D^-1 B) Z_n + D^-1 A = Z_n - D^-1 (B Z_n - A),        niter times.
 * "The individual columns of Z can be computed independently": one column at a time.
 * Z: N x N column-major output (not symmetric in general).
 * ------------------------------------------------------------------------------------------- */
void oracle_eq14_iteration(int64_t N, const double* A, const double* B, int64_t niter, double* Z) {
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < N; ++c) {
        std::vector<double> z(N), r(N);
        for (int64_t i = 0; i < N; ++i) z[i] = A[i + c * N];
        for (int64_t it = 0; it < niter; ++it) {
            for (int64_t i = 0; i < N; ++i) {
                double sum = 0.0;
                for (int64_t k = 0; k < N; ++k) sum += B[i + k * N] * z[k];
                r[i] = sum - A[i + c * N];
            }
            for (int64_t i = 0; i < N; ++i) z[i] -= r[i] / B[i + i * N];
        }
        for (int64_t i = 0; i < N; ++i) Z[i + c * N] = z[i];
    }
}

int oracle_num_threads(void) {
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp single
        n = omp_get_num_threads();
    }
#endif
    return n;
}

} /* extern "C" */
