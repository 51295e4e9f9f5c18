// kernels.cuh -- the non-GEMM kernels of the PFSM path (sm_100a):
//   jacobi_batched_kernel   step 2, second route (option step2_route = 1) for submatrices too large for shared memory: a cluster
//                           of CTAs per slice, one-sided (Hestenes) Jacobi on the slice's shifted submatrix kept in L2,
//                           round-robin parallel ordering, a warp per column pair.  (The product path of step 2 is
//                           tridiag_eig.cuh from M = 16 on, jacobi_smem.cuh below.)
//   chol_diag_kernel        step 4: Cholesky factor + inverse of one 128 x 128 diagonal block
//   extract_diag_kernel     step 4: diag(V^T V) for the breakdown threshold
//   transpose_kernel        step 4: V <-> V^T staging for the stacked Cholesky-QR
//   rayleigh_kernel         step 5: lambda_i = v_i . t_i and r_i = ||t_i - lambda_i v_i||
//   symmetrize_kernel, transpose_blocks_kernel, inv_diag_kernel   row G / Eq. 14 helpers
//   mirror_lower_kernel     pfsm_solve_host: upper block triangle of A from the uploaded lower one
//   fp64 peak probes        roofline calibration
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "gemm_tn.cuh"  // dmma884

namespace pfsm {

struct SliceTable {  // step 1: device-resident, built once in pfsm_create
    const int32_t* g0;   // first global eigen-index of slice s
    const int32_t* lo;   // first row/column of its submatrix
    const int32_t* off;  // local index of the slice's first eigenpair = g0 - lo
    const int32_t* cnt;  // eigenpairs in slice s (N/P, or floor/ceil of it when P does not divide N; reading R14)
};

constexpr int JACOBI_THREADS = 1024;
constexpr int JACOBI_MAX_SWEEPS = 40;

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ---------------------------------------------------------------------------------------------
// Step 2: B_s y = mu y for slice s = blockIdx.x.
//
// One-sided Jacobi on G = B_s + sigma I (sigma = 2 x Gershgorin bound, so G is SPD with condition
// number <= 3): rotate column pairs of G until all columns are mutually orthogonal.  Then
// G = (B_s + sigma I) J with J orthogonal and G^T G diagonal, so column c of G is (mu_c + sigma) y_c:
// the eigenvector is the normalized column and mu_c = ||g_c|| - sigma.  No second matrix is needed.
// G (M x M, column-major, 8 M^2 bytes: 72-512 KiB) lives in the handle's workspace and stays L2
// resident; each warp takes one column pair per turn, holds both columns in registers (EPL doubles
// per lane per column), forms the three dot products with shuffles, rotates and writes back.
// Pairs of a round are disjoint (round-robin tournament), rounds are separated by __syncthreads.
//
// Output: for the slice's m eigenpairs (ascending local ranks off .. off+m-1):
//   eps[g0 + j] = mu;  V[(g0 + j) * N + lo + r] = y[r]   (V was zero-filled before the launch).
// info: atomicMin-style first failure N + s + 1 if the sweep cap is hit.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t cluster_nctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r));
    return r;
}
// barrier over all threads of the cluster's CTAs; release/acquire orders their global-memory accesses
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

// A slice is worked on by a thread-block CLUSTER of CS = 1, 2, 4 or 8 CTAs (launch attribute): the column
// pairs of a tournament round are dealt round-robin to the CS x 32 warps, G stays in L2 (loads bypass L1 with
// ld.global.cg because another SM may have written the column), and the round barrier is the cluster barrier.
// The kernel is bound by L2 bandwidth (every round streams G once), so CS SMs per slice give CS x the L2 ports.
// threads per CTA of the L2-resident kernel: 2 EPL doubles per lane must fit the register file (see jacobi_smem_threads)
__host__ __device__ constexpr int jacobi_l2_threads(int epl) { return epl <= 8 ? JACOBI_THREADS : 512; }

template <int EPL>
__global__ void __launch_bounds__(jacobi_l2_threads(EPL), 1)
jacobi_batched_kernel(const double* __restrict__ A, int64_t N, int32_t M, SliceTable tab,
                      double* __restrict__ Gws, double* __restrict__ V, double* __restrict__ eps,
                      int* __restrict__ rotcnt, unsigned long long* info, int32_t s_off) {
    const int CS = (int)cluster_nctarank(), cr = (int)cluster_ctarank();
    const int s = s_off + blockIdx.x / CS;  // s_off: first slice of this launch (a rank of the sharded solve owns a range)
    const int lo = tab.lo[s], off = tab.off[s], g0 = tab.g0[s], m = tab.cnt[s];
    double* G = Gws + (size_t)s * M * M;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    constexpr int NT = jacobi_l2_threads(EPL), NW = NT / 32;
    const int gw = cr * NW + warp, TW = CS * NW;  // warp index / warp count within the cluster
    int* rot = rotcnt + (size_t)s * JACOBI_MAX_SWEEPS;

    __shared__ double red[NW];
    __shared__ double s_sigma;
    extern __shared__ double dyn[];  // nrm[M] then rank (int) [M]
    double* nrm = dyn;
    int* rank = reinterpret_cast<int*>(dyn + M);

    // Gershgorin bound: max_r sum_c |B[r][c]|  (thread per row; consecutive rows are contiguous).
    // Every CTA of the cluster computes it (same order -> same sigma).
    double bound = 0.0;
    for (int r = tid; r < M; r += NT) {
        double sum = 0.0;
        for (int c = 0; c < M; ++c) sum += fabs(A[(size_t)(lo + c) * N + lo + r]);
        bound = fmax(bound, sum);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) bound = fmax(bound, __shfl_xor_sync(0xffffffffu, bound, o));
    if (lane == 0) red[warp] = bound;
    __syncthreads();
    if (tid == 0) {
        double b = 0.0;
        for (int w = 0; w < NW; ++w) b = fmax(b, red[w]);
        s_sigma = (b > 0.0) ? 2.0 * b : 1.0;
    }
    __syncthreads();
    const double sigma = s_sigma;
    for (int idx = cr * NT + tid; idx < M * M; idx += CS * NT) {
        const int c = idx / M, r = idx - c * M;
        double v = A[(size_t)(lo + c) * N + lo + r];
        if (r == c) v += sigma;
        G[idx] = v;
    }
    cluster_sync_all();

    const int Me = M + (M & 1);  // phantom column when M is odd
    const int n1 = Me - 1, npairs = Me / 2;
    const double tol = 2.220446049250313e-16 * sqrt((double)M);
    bool converged = false;
    for (int sweep = 0; sweep < JACOBI_MAX_SWEEPS; ++sweep) {
        int nrot = 0;
        for (int rnd = 0; rnd < n1; ++rnd) {
            for (int pi = gw; pi < npairs; pi += TW) {
                int p, q;
                if (pi == 0) {
                    p = n1;
                    q = rnd;
                } else {
                    p = rnd + pi;
                    if (p >= n1) p -= n1;
                    q = rnd - pi;
                    if (q < 0) q += n1;
                }
                if (p >= M || q >= M) continue;
                if (p > q) {
                    const int tmp = p;
                    p = q;
                    q = tmp;
                }
                double* gp = G + (size_t)p * M;
                double* gq = G + (size_t)q * M;
                double x[EPL], y[EPL];
                double aa = 0.0, bb = 0.0, ab = 0.0;
#pragma unroll
                for (int e = 0; e < EPL; ++e) {
                    const int r = lane + 32 * e;
                    x[e] = (r < M) ? __ldcg(gp + r) : 0.0;
                    y[e] = (r < M) ? __ldcg(gq + r) : 0.0;
                    aa = fma(x[e], x[e], aa);
                    bb = fma(y[e], y[e], bb);
                    ab = fma(x[e], y[e], ab);
                }
                aa = warp_sum(aa);
                bb = warp_sum(bb);
                ab = warp_sum(ab);
                if (fabs(ab) > tol * sqrt(aa * bb)) {
                    const double zeta = (bb - aa) / (2.0 * ab);
                    const double tt = copysign(1.0, zeta) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
                    const double cs = 1.0 / sqrt(1.0 + tt * tt), sn = cs * tt;
#pragma unroll
                    for (int e = 0; e < EPL; ++e) {
                        const int r = lane + 32 * e;
                        if (r < M) {
                            gp[r] = cs * x[e] - sn * y[e];
                            gq[r] = sn * x[e] + cs * y[e];
                        }
                    }
                    ++nrot;
                }
            }
            if (rnd == n1 - 1 && lane == 0 && nrot) atomicAdd(rot + sweep, nrot);
            cluster_sync_all();
        }
        const int total = __ldcg(rot + sweep);
        if (total == 0) {
            converged = true;
            break;
        }
    }
    if (!converged && tid == 0 && cr == 0) atomicMin(info, (unsigned long long)(N + s + 1));

    // column norms -> eigenvalues; rank by counting (ties: lower column index first)
    for (int c = warp; c < M; c += NW) {
        const double* gc = G + (size_t)c * M;
        double ss = 0.0;
        for (int r = lane; r < M; r += 32) {
            const double g = __ldcg(gc + r);
            ss = fma(g, g, ss);
        }
        ss = warp_sum(ss);
        if (lane == 0) nrm[c] = sqrt(ss);
    }
    __syncthreads();
    for (int c = tid; c < M; c += NT) {
        const double v = nrm[c];
        int rk = 0;
        for (int j = 0; j < M; ++j) {
            const double u = nrm[j];
            rk += (u < v || (u == v && j < c)) ? 1 : 0;
        }
        rank[c] = rk;
    }
    __syncthreads();
    for (int c = gw; c < M; c += TW) {
        const int j = rank[c] - off;
        if (j < 0 || j >= m) continue;
        const double nv = nrm[c];
        const double inv = 1.0 / nv;
        const double* gc = G + (size_t)c * M;
        double* v = V + (size_t)(g0 + j) * N + lo;
        // sign convention: largest-magnitude component positive is not needed (R16); keep G's sign
        for (int r = lane; r < M; r += 32) v[r] = __ldcg(gc + r) * inv;
        if (lane == 0) eps[g0 + j] = nv - sigma;
    }
}

// ---------------------------------------------------------------------------------------------
// Step 4 helper: Cholesky factor and inverse of one diagonal block (order nb <= 128) of the stacked
// matrix S (row-major view, leading dimension ld).  Reads the lower triangle of S[k0:k0+nb, k0:k0+nb],
// writes L (lower, upper zeroed) to Lout[k0:k0+nb, k0:k0+nb] (leading dimension ld) and L^-1 (lower,
// zero padded to 128 x 128) to Dinv (leading dimension 128).  A non-positive pivot j sets
// info = min(info, k0 + j + 1) (the vectors are numerically dependent).
// ---------------------------------------------------------------------------------------------
constexpr int CHOL_NB = 128;
constexpr int CHOL_THREADS = 1024;
constexpr int CHOL_LDS = CHOL_NB + 1;
constexpr int CHOL_SMEM = (CHOL_NB * CHOL_LDS + 3 * CHOL_NB + 64 * 64) * 8;  // L below, L^-1 (transposed) above the diagonal

// diag(G) before the factorization: the breakdown test compares each pivot with its original diagonal entry
__global__ void extract_diag_kernel(const double* __restrict__ S, int64_t ld, int32_t n, double* __restrict__ gdiag) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) gdiag[i] = S[(size_t)i * ld + i];
}

// dinv[i] = 1 / B[i][i]  (Eq. 14: D = diag(B))
__global__ void inv_diag_kernel(const double* __restrict__ B, int64_t ld, int32_t n, double* __restrict__ dinv) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dinv[i] = 1.0 / B[(size_t)i * ld + i];
}

// A pivot counts as "not positive" when it is <= CHOL_BREAKDOWN * (its original diagonal entry ||v_j||^2):
// below that the projected vector has lost 6 digits to its predecessors and single-pass Cholesky-QR
// (orthogonality error ~ eps * cond(V)^2) can no longer deliver orthonormal vectors.
constexpr double CHOL_BREAKDOWN = 1e-12;

// Blocked in 16-wide panels so that only 3 block barriers per panel (24 in all) sit on the serial chain:
//   A1 warp 0 factors the 16 x 16 diagonal block (lane = row, __syncwarp between columns)
//   A2 one thread per row below solves its 16 entries against that block
//   A3 all threads apply the rank-16 update to the trailing lower triangle
// then L^-1: B1 eight warps invert the 16 x 16 diagonal blocks, B2 recursive doubling (b = 16, 32, 64) joins adjacent
// inverted blocks.  The rank-16 updates of A3 and the products of B2 run on the FP64 tensor pipe (DMMA).
// Rows/columns >= nb are padded with the identity and masked on output.
__global__ void __launch_bounds__(CHOL_THREADS, 1)
chol_diag_kernel(const double* __restrict__ S, double* __restrict__ Lout, int64_t ld, int32_t k0, int32_t nb,
                 double* __restrict__ Dinv, const double* __restrict__ gdiag, unsigned long long* info) {
    extern __shared__ double sm[];
    // a[i][c] (leading dimension CHOL_LDS): c <= i holds L; the strictly upper part holds the strictly
    // lower part of L^-1 transposed (L^-1[r][c] at a[c][r], r > c); idiag[c] = 1 / L[c][c] = L^-1[c][c].
    double* a = sm;
    double* idiag = sm + CHOL_NB * CHOL_LDS;
    double* T = idiag + CHOL_NB;  // 64 x 64 scratch of phase B2
    double* thr = T + 64 * 64;    // breakdown threshold per column (0 for padding columns)
    double* ldiag = thr + CHOL_NB;  // L's diagonal while `a`'s diagonal holds L^-1's
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    {   // all 16 loads of a thread are issued before the first use (clamped addresses, masked afterwards)
        double v[CHOL_NB * CHOL_NB / CHOL_THREADS];
#pragma unroll
        for (int q = 0; q < CHOL_NB * CHOL_NB / CHOL_THREADS; ++q) {
            const int idx = tid + q * CHOL_THREADS, i = idx >> 7, c = idx & 127;
            v[q] = S[(size_t)(k0 + min(i, nb - 1)) * ld + k0 + min(c, nb - 1)];
        }
#pragma unroll
        for (int q = 0; q < CHOL_NB * CHOL_NB / CHOL_THREADS; ++q) {
            const int idx = tid + q * CHOL_THREADS, i = idx >> 7, c = idx & 127;
            a[i * CHOL_LDS + c] = (i < nb && c < nb) ? (c <= i ? v[q] : 0.0) : (i == c ? 1.0 : 0.0);
        }
    }
    if (tid < CHOL_NB) thr[tid] = (tid < nb) ? CHOL_BREAKDOWN * gdiag[k0 + tid] : 0.0;
    __syncthreads();

    // ---------------- phase A: L ----------------
    for (int j0 = 0; j0 < CHOL_NB; j0 += 16) {
        if (warp == 0) {
            // A1: the 16 x 16 diagonal block in registers, lane = row (lanes 16..31 carry zeros), columns exchanged
            // with shuffles; fully unrolled, no shared-memory round trips on the serial chain.
            const int i = j0 + (lane & 15);
            double r[16];
#pragma unroll
            for (int c = 0; c < 16; ++c) r[c] = (lane < 16 && c <= lane) ? a[i * CHOL_LDS + j0 + c] : 0.0;
#pragma unroll
            for (int j = 0; j < 16; ++j) {
                double piv = __shfl_sync(0xffffffffu, r[j], j);
                if (!(piv > thr[j0 + j]) || !(piv > 0.0)) {
                    if (lane == 0) atomicMin(info, (unsigned long long)(k0 + j0 + j + 1));
                    piv = 1.0;
                }
                const double rd = rsqrt(piv);  // (1 ulp; the scaling below sits on the serial chain, so no refinement there)
                double d = piv * rd;
                d = fma(fma(-d, d, piv), 0.5 * rd, d);  // off the chain: d = sqrt(piv) to the last bit or two (only lane j keeps it)
                r[j] = (lane == j) ? d : r[j] * rd;
                if (lane == j) idiag[j0 + j] = rd;
#pragma unroll
                for (int c = j + 1; c < 16; ++c) {
                    const double lc = __shfl_sync(0xffffffffu, r[j], c);  // l[c][j]
                    r[c] = fma(-r[j], lc, r[c]);                          // meaningful for lanes >= c
                }
            }
            if (lane < 16) {
#pragma unroll
                for (int c = 0; c < 16; ++c)
                    if (c <= lane) a[i * CHOL_LDS + j0 + c] = r[c];
            }
        }
        __syncthreads();
        if (j0 + 16 >= CHOL_NB) break;
        if (tid < CHOL_NB && tid >= j0 + 16) {  // A2: row tid of the panel
            const int i = tid;
            double x[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) {
                double s = a[i * CHOL_LDS + j0 + j];
#pragma unroll
                for (int k = 0; k < j; ++k) s -= x[k] * a[(j0 + j) * CHOL_LDS + j0 + k];
                x[j] = s * idiag[j0 + j];
            }
#pragma unroll
            for (int j = 0; j < 16; ++j) a[i * CHOL_LDS + j0 + j] = x[j];
        }
        __syncthreads();
        {  // A3: a[i][c] -= sum_k l[i][k] l[c][k] on the trailing lower triangle, on the FP64 tensor pipe: one
           // 16 x 16 block per warp (at most 28 lower blocks), K = 16 = four DMMA k-steps.  The part of a diagonal
           // block above the diagonal gets updated too; nothing reads it before phase B overwrites it.
            const int nbk = (CHOL_NB - j0 - 16) / 16;
            if (warp < nbk * (nbk + 1) / 2) {
                int bi = 0;
                while ((bi + 1) * (bi + 2) / 2 <= warp) ++bi;
                const int bj = warp - bi * (bi + 1) / 2;
                const int i0 = j0 + 16 + 16 * bi, c0 = j0 + 16 + 16 * bj;
                const int g = lane >> 2, t = lane & 3;
                double acc[2][2][2] = {{{0.0, 0.0}, {0.0, 0.0}}, {{0.0, 0.0}, {0.0, 0.0}}};
#pragma unroll
                for (int k = 0; k < 16; k += 4) {
                    const double x0 = a[(i0 + g) * CHOL_LDS + j0 + k + t], x1 = a[(i0 + 8 + g) * CHOL_LDS + j0 + k + t];
                    const double y0 = a[(c0 + g) * CHOL_LDS + j0 + k + t], y1 = a[(c0 + 8 + g) * CHOL_LDS + j0 + k + t];
                    dmma884(acc[0][0][0], acc[0][0][1], x0, y0);
                    dmma884(acc[0][1][0], acc[0][1][1], x0, y1);
                    dmma884(acc[1][0][0], acc[1][0][1], x1, y0);
                    dmma884(acc[1][1][0], acc[1][1][1], x1, y1);
                }
#pragma unroll
                for (int ri = 0; ri < 2; ++ri)
#pragma unroll
                    for (int ci = 0; ci < 2; ++ci) {
                        double* cp = a + (i0 + 8 * ri + g) * CHOL_LDS + c0 + 8 * ci + 2 * t;
                        cp[0] -= acc[ri][ci][0];
                        cp[1] -= acc[ri][ci][1];
                    }
            }
        }
        __syncthreads();
    }

    // ---------------- phase B: L^-1 ----------------
    if (warp < 8 && lane < 16) {  // B1: diagonal block `warp`, column `lane` by forward substitution
        const int b0 = warp * 16, c = lane;
        for (int r = c + 1; r < 16; ++r) {
            double s = a[(b0 + r) * CHOL_LDS + b0 + c] * idiag[b0 + c];
            for (int k = c + 1; k < r; ++k) s = fma(a[(b0 + r) * CHOL_LDS + b0 + k], a[(b0 + c) * CHOL_LDS + b0 + k], s);
            a[(b0 + c) * CHOL_LDS + b0 + r] = -s * idiag[b0 + r];
        }
    }
    __syncthreads();
    // From here on the diagonal of `a` holds L^-1's diagonal (L's goes to ldiag), so L^-1[x][y] for x >= y is
    // uniformly a[y][x] (transposed storage).
    if (tid < CHOL_NB) {
        ldiag[tid] = a[tid * CHOL_LDS + tid];
        a[tid * CHOL_LDS + tid] = idiag[tid];
    }
    __syncthreads();
    // B2: recursive doubling on the FP64 tensor pipe.  With the inverses A^-1, B^-1 of two adjacent b x b diagonal
    // blocks known,  [A 0; C B]^-1 = [A^-1 0; -B^-1 C A^-1  B^-1];  b = 16, 32, 64: three levels, each two products,
    // one 16 x 16 output block per warp (4, 8, 16 warps), fragments gathered straight from the (transposed) storage.
    {
        const int g = lane >> 2, t = lane & 3;
        for (int b = 16, lb = 4; b < CHOL_NB; b *= 2, ++lb) {
            const int n16 = b >> 4, bpp = n16 * n16, total = (CHOL_NB / (2 * b)) * bpp;
            const int pr = warp / bpp, rem = warp - pr * bpp, bi = rem / n16, bj = rem - bi * n16;
            const int o = pr * 2 * b, i0 = 16 * bi, j0 = 16 * bj;
            double* Tp = T + (pr << (2 * lb));  // T of this pair, b x b row-major
            if (warp < total) {  // T = C A^-1:  T[i][j] = sum_{k >= j} C[i][k] A^-1[k][j]
                double acc[2][2][2] = {{{0.0, 0.0}, {0.0, 0.0}}, {{0.0, 0.0}, {0.0, 0.0}}};
                for (int kb = bj; kb < n16; ++kb) {
#pragma unroll
                    for (int k4 = 0; k4 < 16; k4 += 4) {
                        const int k = 16 * kb + k4 + t;
                        const double x0 = a[(o + b + i0 + g) * CHOL_LDS + o + k], x1 = a[(o + b + i0 + 8 + g) * CHOL_LDS + o + k];
                        double y0 = a[(o + j0 + g) * CHOL_LDS + o + k], y1 = a[(o + j0 + 8 + g) * CHOL_LDS + o + k];
                        if (k < j0 + g) y0 = 0.0;      // A^-1[k][j] = 0 for k < j (the storage holds L there)
                        if (k < j0 + 8 + g) y1 = 0.0;
                        dmma884(acc[0][0][0], acc[0][0][1], x0, y0);
                        dmma884(acc[0][1][0], acc[0][1][1], x0, y1);
                        dmma884(acc[1][0][0], acc[1][0][1], x1, y0);
                        dmma884(acc[1][1][0], acc[1][1][1], x1, y1);
                    }
                }
#pragma unroll
                for (int ri = 0; ri < 2; ++ri)
#pragma unroll
                    for (int ci = 0; ci < 2; ++ci) {
                        double* tp = Tp + ((i0 + 8 * ri + g) << lb) + j0 + 8 * ci + 2 * t;
                        tp[0] = acc[ri][ci][0];
                        tp[1] = acc[ri][ci][1];
                    }
            }
            __syncthreads();
            if (warp < total) {  // out^T[j][i] = -sum_{k <= i} T[k][j] B^-1[i][k], stored at a[o+j][o+b+i]
                double acc[2][2][2] = {{{0.0, 0.0}, {0.0, 0.0}}, {{0.0, 0.0}, {0.0, 0.0}}};
                for (int kb = 0; kb <= bi; ++kb) {
#pragma unroll
                    for (int k4 = 0; k4 < 16; k4 += 4) {
                        const int k = 16 * kb + k4 + t;
                        const double x0 = Tp[(k << lb) + j0 + g], x1 = Tp[(k << lb) + j0 + 8 + g];
                        double y0 = a[(o + b + k) * CHOL_LDS + o + b + i0 + g], y1 = a[(o + b + k) * CHOL_LDS + o + b + i0 + 8 + g];
                        if (k > i0 + g) y0 = 0.0;      // B^-1[i][k] = 0 for k > i
                        if (k > i0 + 8 + g) y1 = 0.0;
                        dmma884(acc[0][0][0], acc[0][0][1], x0, y0);
                        dmma884(acc[0][1][0], acc[0][1][1], x0, y1);
                        dmma884(acc[1][0][0], acc[1][0][1], x1, y0);
                        dmma884(acc[1][1][0], acc[1][1][1], x1, y1);
                    }
                }
#pragma unroll
                for (int ri = 0; ri < 2; ++ri)      // tile rows = j, tile columns = i
#pragma unroll
                    for (int ci = 0; ci < 2; ++ci) {
                        double* op = a + (o + j0 + 8 * ri + g) * CHOL_LDS + o + b + i0 + 8 * ci + 2 * t;
                        op[0] = -acc[ri][ci][0];
                        op[1] = -acc[ri][ci][1];
                    }
            }
            __syncthreads();
        }
    }
#pragma unroll 4
    for (int idx = tid; idx < CHOL_NB * CHOL_NB; idx += CHOL_THREADS) {
        const int r = idx >> 7, c = idx & 127;
        const bool in = (r < nb && c < nb);
        Dinv[idx] = (in && c <= r) ? a[c * CHOL_LDS + r] : 0.0;
        if (in) Lout[(size_t)(k0 + r) * ld + k0 + c] = (c < r) ? a[r * CHOL_LDS + c] : (c == r ? ldiag[r] : 0.0);
    }
}

// out[c][r] = in[r][c] for an nr x nc row-major matrix (leading dimensions ldi / ldo)
__global__ void transpose_kernel(const double* __restrict__ in, int64_t ldi, double* __restrict__ out,
                                 int64_t ldo, int32_t nr, int32_t nc) {
    __shared__ double tile[32][33];
    const int bx = blockIdx.x * 32, by = blockIdx.y * 32;
    const int tx = threadIdx.x, ty = threadIdx.y;  // 32 x 8
#pragma unroll
    for (int k = 0; k < 32; k += 8) {
        const int r = by + ty + k, c = bx + tx;
        if (r < nr && c < nc) tile[ty + k][tx] = in[(size_t)r * ldi + c];
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 32; k += 8) {
        const int c = bx + ty + k, r = by + tx;
        if (r < nr && c < nc) out[(size_t)c * ldo + r] = tile[tx][ty + k];
    }
}

// Fills the block-upper part of a symmetric matrix from its block-lower part: for 32 x 32 tiles whose column lies in
// a later RB-row block than their row, out tile (r, c) = transpose of tile (c, r).  pfsm_solve_host uploads only the
// lower block triangle of A (half the PCIe bytes) and mirrors it here.  RB must be a multiple of 32.
__global__ void mirror_lower_kernel(double* __restrict__ A, int64_t ld, int32_t n, int32_t RB) {
    __shared__ double tile[32][33];
    const int bx = blockIdx.x * 32, by = blockIdx.y * 32;  // destination tile: rows by.., columns bx..
    if (bx / RB <= by / RB) return;
    const int tx = threadIdx.x, ty = threadIdx.y;  // 32 x 8
#pragma unroll
    for (int k = 0; k < 32; k += 8) {
        const int r = bx + ty + k, c = by + tx;  // source tile: rows bx.., columns by..
        if (r < n && c < n) tile[ty + k][tx] = A[(size_t)r * ld + c];
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 32; k += 8) {
        const int r = by + ty + k, c = bx + tx;
        if (r < n && c < n) A[(size_t)r * ld + c] = tile[tx][ty + k];
    }
}

// out = (in + in^T) / 2 for an n x n row-major matrix (32 x 32 tiles, both reads coalesced)
__global__ void symmetrize_kernel(const double* __restrict__ in, int64_t ldi, double* __restrict__ out, int64_t ldo,
                                  int32_t n) {
    __shared__ double t1[32][33], t2[32][33];
    const int bx = blockIdx.x * 32, by = blockIdx.y * 32;
    const int tx = threadIdx.x, ty = threadIdx.y;  // 32 x 8
#pragma unroll
    for (int k = 0; k < 32; k += 8) {
        const int r = by + ty + k, c = bx + tx;
        t1[ty + k][tx] = (r < n && c < n) ? in[(size_t)r * ldi + c] : 0.0;
        const int r2 = bx + ty + k, c2 = by + tx;
        t2[ty + k][tx] = (r2 < n && c2 < n) ? in[(size_t)r2 * ldi + c2] : 0.0;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 32; k += 8) {
        const int r = by + ty + k, c = bx + tx;
        if (r < n && c < n) out[(size_t)r * ldo + c] = 0.5 * (t1[ty + k][tx] + t2[tx][ty + k]);
    }
}

// out block b = transpose of in block b, for nblocks dense 128 x 128 blocks (grid: 4 x 4 x nblocks, block 32 x 8)
__global__ void transpose_blocks_kernel(const double* __restrict__ in, double* __restrict__ out) {
    __shared__ double tile[32][33];
    const size_t base = (size_t)blockIdx.z * 128 * 128;
    const int bx = blockIdx.x * 32, by = blockIdx.y * 32;
    const int tx = threadIdx.x, ty = threadIdx.y;
#pragma unroll
    for (int k = 0; k < 32; k += 8) tile[ty + k][tx] = in[base + (size_t)(by + ty + k) * 128 + bx + tx];
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 32; k += 8) out[base + (size_t)(bx + ty + k) * 128 + by + tx] = tile[tx][ty + k];
}

// ---------------------------------------------------------------------------------------------
// Step 5: one CTA per eigenvector i.  lambda_i = v_i . t_i  (t_i = A v_i from the GEMM), then
// r_i = || t_i - lambda_i v_i ||_2.  Vectorised, coalesced; fixed reduction order (deterministic).
// ---------------------------------------------------------------------------------------------
constexpr int RAY_THREADS = 256;
__device__ __forceinline__ double block_sum(double v, double* red) {
    v = warp_sum(v);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();
    if (lane == 0) red[warp] = v;
    __syncthreads();
    double t = 0.0;
    for (int w = 0; w < RAY_THREADS / 32; ++w) t += red[w];
    return t;
}
__global__ void __launch_bounds__(RAY_THREADS)
rayleigh_kernel(const double* __restrict__ V, const double* __restrict__ T, int64_t ld, int64_t N, double* __restrict__ lambda,
                double* __restrict__ resid, int32_t i_off) {
    __shared__ double red[RAY_THREADS / 32];
    const int64_t i = (int64_t)i_off + blockIdx.x;
    const double2* v2 = reinterpret_cast<const double2*>(V + i * ld);  // ld is even: rows are 16-byte aligned
    const double2* t2 = reinterpret_cast<const double2*>(T + i * ld);
    const int64_t n2 = N / 2;
    const bool tail = (N & 1) && threadIdx.x == 0;  // odd N: the last component, by thread 0
    const double vt = tail ? V[i * ld + N - 1] : 0.0, tt = tail ? T[i * ld + N - 1] : 0.0;
    double s = vt * tt;
#pragma unroll 4
    for (int64_t k = threadIdx.x; k < n2; k += RAY_THREADS) {
        const double2 a = v2[k], b = t2[k];
        s = fma(a.x, b.x, s);
        s = fma(a.y, b.y, s);
    }
    const double lam = block_sum(s, red);
    const double et = tt - lam * vt;
    double q = et * et;
#pragma unroll 4
    for (int64_t k = threadIdx.x; k < n2; k += RAY_THREADS) {
        const double2 a = v2[k], b = t2[k];
        const double e0 = b.x - lam * a.x, e1 = b.y - lam * a.y;
        q = fma(e0, e0, q);
        q = fma(e1, e1, q);
    }
    const double rr = block_sum(q, red);
    if (threadIdx.x == 0) {
        lambda[i] = lam;
        resid[i] = sqrt(rr);
    }
}

// Peer-write mode of the sharded solve: copies `count` doubles of this rank's result into the same place of every other
// rank's buffer (peer device memory mapped through CUDA IPC).  Used for what no GEMM epilogue produces: lambda and the
// residuals (N / world doubles each), and the start vectors when there are no folded-spectrum iterations.
struct PeerPtrs {
    double* p[GEMM_MAX_PEERS];
    int32_t n;
};
__global__ void peer_copy_kernel(const double* __restrict__ src, int64_t count, PeerPtrs dst) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (int64_t)gridDim.x * blockDim.x) {
        const double v = src[i];
        for (int q = 0; q < dst.n; ++q) dst.p[q][i] = v;
    }
    __threadfence_system();
}

// max_i r[i] (NaN counts as +inf) -> out[0]; one CTA, fixed order.  The validity guard of PAPER.md:98-100.
__global__ void __launch_bounds__(1024) max_residual_kernel(const double* __restrict__ r, int64_t N, double* __restrict__ out) {
    __shared__ double red[32];
    double m = 0.0;
    for (int64_t i = threadIdx.x; i < N; i += 1024) {
        const double v = r[i];
        m = fmax(m, (v == v) ? v : __longlong_as_double(0x7ff0000000000000LL));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < 32; ++w) t = fmax(t, red[w]);
        out[0] = t;
    }
}

// ---------------------------------------------------------------------------------------------
// Roofline calibration: register-only FP64 issue-rate loops (no memory traffic).
// ---------------------------------------------------------------------------------------------
// 4 accumulator pairs per warp, reused in place (with 16 ptxas emits out-of-place DMMAs whose WAW hazards
// stall the pipe and the loop reads ~20 % low); 8 warps per SMSP hide the DMMA latency.
__global__ void __launch_bounds__(256) probe_dmma_kernel(int iters, double* sink) {
    double c[4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i) c[i][0] = c[i][1] = 0.0;
    const double a = 1.0 + 1e-9 * threadIdx.x, b = 1.0 - 1e-9 * threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int i = 0; i < 4; ++i)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                             : "+d"(c[i][0]), "+d"(c[i][1])
                             : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 4; ++i) s += c[i][0] + c[i][1];
    if (s == 123.456) sink[0] = s;
}
__global__ void __launch_bounds__(256) probe_dfma_kernel(int iters, double* sink) {
    double c[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) c[i] = 1e-3 * i;
    const double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-9 * threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(c[i]) : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += c[i];
    if (s == 123.456) sink[0] = s;
}

}  // namespace pfsm
