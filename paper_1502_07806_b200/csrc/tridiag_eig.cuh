// tridiag_eig.cuh -- step 2 as a batched dense symmetric eigensolver in five kernels: the product path for
// submatrix orders 16 <= M <= 8192, i.e. all BASELINE configs (M = 96-256) and the paper's wide windows (gamma = M/N = 0.2-0.3,
// "M <= 3000").  Only the slice's m of the M eigenpairs of B_s are wanted (local ascending ranks
// off .. off+m-1), which this route exploits:
//
//   sytrd_kernel<CLUSTER>   B_s = Q T Q^T, Householder tridiagonalization of all slices at once on full symmetric storage.  The
//                           rank-2 update of column k-1 is applied inside the pass that forms the matrix-vector product of
//                           column k, so the trailing matrix is read and written once per column (16 (M-k)^2 bytes).
//                           CLUSTER (M <= 768): one thread-block cluster per slice, cluster barrier per column -- latency bound;
//                           otherwise ONE persistent cooperative grid, C CTAs per slice, grid barrier per column.
//   sytrd_dsmem_kernel      the same with the submatrix resident in the distributed shared memory of the slice's cluster: the
//                           default for small M (all BASELINE configs), no global-memory access on the per-column chain
//   (sytrd_blocked.cuh)     the blocked variant with DMMA trailing updates: the default once the batch is well beyond L2
//   sytrd_half_kernel       the same on the lower triangle only (half the bytes, two grid barriers per column): used when the
//                           batch 8 P M^2 exceeds L2, where the tridiagonalization is HBM bound
//   tri_bisect_kernel       eigenvalue of rank off+t of T by 33-way multi-section on the Sturm count, one warp per eigenvalue
//   tri_invit_kernel        its eigenvector by inverse iteration: LU of T - lambda I with partial pivoting, three
//                           solves from a counter-based random start, one thread per eigenvector, factors stored
//                           [row][vector] so that a warp's accesses coalesce
//   tri_cluster_kernel      re-orthogonalization + re-iteration inside eigenvalue clusters tighter than 1e-7 ||T|| (dstein's scheme)
//   tri_backtransform_kernel  y = H_0 H_1 ... H_{M-3} z, eight (four, two) eigenvectors per CTA held in registers, each
//                           reflector read once per CTA, written zero-padded into V
//
// Eigenvalues closer than 10 eps max(|lambda|, 1e-3 ||T||) get shifts pushed apart as LAPACK's dstein does; vectors of runs
// of eigenvalues closer than 1e-7 ||T|| are re-orthogonalized and re-iterated (tri_cluster_kernel); wider gaps leave at most
// 2e-9 of non-orthogonality, which step 4 removes (it orthonormalizes all N vectors anyway).  A vector whose
// last solve did not converge flags its slice (info = N + s + 1).
// Every reduction has a fixed order: results are bitwise reproducible.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "jacobi_wide.cuh"  // jw_grid_barrier
#include "kernels.cuh"

namespace pfsm {

constexpr int TRD_THREADS = 512;
constexpr int TRI_THREADS = 128;  // bisection / inverse iteration: threads (= eigenpairs) per CTA

struct TriWs {                  // workspace of the tridiagonal route (device pointers)
    double* d;                  // P x M   diagonal of T
    double* e;                  // P x M   sub-diagonal of T (e[k] couples k and k+1)
    double* tau;                // P x M   Householder scalars
    double* pbuf;               // 2 x P x M   matrix-vector products, double-buffered by column parity
    double* vbuf;               // 2 x P x M   current Householder vector, double-buffered
    double* rowbuf;             // P x ceil(M/32) x M   row-part partial sums of the half-storage product
    double* colbuf;             // P x ceil(M/32) x M   column-part partial sums
    double* colk;               // 2 x P x M   column k+1 of the trailing matrix, written by the pass of column k
    double* lam;                // N       eigenvalues (unperturbed)
    double* zscale;             // N       1 / ||z|| of the inverse-iteration vector
    double* f[5];               // 5 x (M x N): U diagonal reciprocal, U super-diagonals 1 and 2, L multipliers, z
    unsigned char* piv;         // M x N   row interchange flags
};

__device__ __forceinline__ double block_sum_512(double v, double* red) {  // fixed order -> every CTA gets the same bits
    v = warp_sum(v);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
#pragma unroll
    for (int w = 0; w < TRD_THREADS / 32; ++w) s += red[w];
    return s;
}

// ---------------------------------------------------------------------------------------------
// Householder tridiagonalization (the unblocked LAPACK dsytd2 recurrence, lower variant, on full symmetric storage).
// Virtual CTA (sl, c), c < C, owns rows i with i % C == c of slice s_off + sl.  Column k:
//   prologue (every CTA of the slice, redundantly and bitwise identically):
//     w_{k-1} = p_{k-1} - (tau_{k-1}/2)(p_{k-1} . v_{k-1}) v_{k-1}            (p from pbuf, v from vbuf)
//     column k of the updated matrix: cc = B[k, k:] - (v_{k-1} w_{k-1}[k] + w_{k-1} v_{k-1}[k]);  d[k] = cc[k]
//     Householder vector of cc[k+1:]: beta = -sign(alpha) ||x||, tau = (beta - alpha)/beta, v = x/(alpha - beta), v[k+1] = 1
//   pass (owned rows i > k): B[i, k+1:] -= v_{k-1}[i] w_{k-1} + w_{k-1}[i] v_{k-1};  p_k[i] = tau_k B[i, k+1:] . v_k
//   grid barrier.
// Reflector k is kept in row k of the slice's matrix (columns k+1 .., leading 1 stored) once that row is dead.
// ---------------------------------------------------------------------------------------------
// CLUSTER: the C CTAs of a slice form one thread-block cluster (grid = ns * C, no cooperative launch) and synchronize
// with the hardware cluster barrier instead of the grid-wide counter -- slices are independent, and for the small
// submatrices of the BASELINE configs a column is latency bound (M = 256, P = 64: 13.7 -> ~5 us per column).
template <bool CLUSTER>
__global__ void __launch_bounds__(TRD_THREADS, 2)
sytrd_kernel(const double* __restrict__ A, int64_t N, int32_t M, SliceTable tab, double* __restrict__ Gws, TriWs ws,
             int32_t P, int32_t s_off, int32_t ns, int32_t C, unsigned int* __restrict__ bar, int32_t precopied) {
    extern __shared__ double sm[];
    double* vp = sm;          // v_{k-1}
    double* wp = sm + M;      // w_{k-1}
    double* vn = sm + 2 * M;  // v_k
    __shared__ double red[TRD_THREADS / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = TRD_THREADS / 32;
    unsigned int phase = 0;
    const int nv = ns * C;

    // copy B_s (row lo + i of A, columns lo ..) into the workspace, unless pfsm_solve_host uploaded the blocks there
    for (int vb = blockIdx.x; vb < nv && !precopied; vb += gridDim.x) {
        const int sl = vb / C, c = vb - sl * C, s = s_off + sl;
        const int lo = tab.lo[s];
        double* G = Gws + (size_t)s * M * M;
        for (int i = c + C * warp; i < M; i += C * NW) {
            const double* a = A + (size_t)(lo + i) * N + lo;
            for (int j = lane; j < M; j += 32) G[(size_t)i * M + j] = a[j];
        }
    }
    if (CLUSTER) cluster_sync_all(); else jw_grid_barrier(bar, phase);

    for (int k = 0; k <= M - 2; ++k) {
        for (int vb = blockIdx.x; vb < nv; vb += gridDim.x) {
            const int sl = vb / C, c = vb - sl * C, s = s_off + sl;
            double* G = Gws + (size_t)s * M * M;
            const size_t so = (size_t)s * M;
            __syncthreads();  // shared vectors of the previous virtual CTA are no longer read
            // ---- prologue (row k is requested first so that its latency overlaps the p / v loads)
            double bk[8];  // M <= 4096 = 8 x 512
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const int i = k + tid + TRD_THREADS * e;
                bk[e] = (i < M) ? __ldcg(G + (size_t)k * M + i) : 0.0;
            }
            double tau_p = 0.0;
            if (k > 0) {
                tau_p = __ldcg(ws.tau + so + k - 1);
                const double* pv_ = ws.pbuf + (size_t)((k - 1) & 1) * P * M + so;
                const double* vv_ = ws.vbuf + (size_t)((k - 1) & 1) * P * M + so;
                double acc = 0.0;
                for (int i = k + tid; i < M; i += TRD_THREADS) {
                    const double v = __ldcg(vv_ + i), p = __ldcg(pv_ + i);
                    vp[i] = v;
                    wp[i] = p;
                    acc = fma(p, v, acc);
                }
                const double pv = block_sum_512(acc, red);
                const double hf = 0.5 * tau_p * pv;
                for (int i = k + tid; i < M; i += TRD_THREADS) wp[i] = fma(-hf, vp[i], wp[i]);
                __syncthreads();
                if (c == 0)  // row k-1 is dead: keep reflector k-1 there (columns k .., leading 1 included)
                    for (int i = k + tid; i < M; i += TRD_THREADS) G[(size_t)(k - 1) * M + i] = vp[i];
            }
            double acc = 0.0, alpha = 0.0, dk = 0.0;
            {
                const double wk = (k > 0) ? wp[k] : 0.0, vk = (k > 0) ? vp[k] : 0.0;
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int i = k + tid + TRD_THREADS * e;
                    if (i < M) {
                        double b = bk[e];
                        if (k > 0) b -= (__dmul_rn(vp[i], wk) + __dmul_rn(wp[i], vk));
                        vn[i] = b;
                        if (i >= k + 2) acc = fma(b, b, acc);
                    }
                }
            }
            const double xn2 = block_sum_512(acc, red);  // (its barriers also publish vn)
            dk = vn[k];
            alpha = vn[k + 1];
            double tau = 0.0, beta = alpha, scal = 0.0;
            if (xn2 > 0.0) {
                beta = -copysign(sqrt(fma(alpha, alpha, xn2)), alpha);
                tau = (beta - alpha) / beta;
                scal = 1.0 / (alpha - beta);
            }
            __syncthreads();
            for (int i = k + 1 + tid; i < M; i += TRD_THREADS) vn[i] = (i == k + 1) ? 1.0 : vn[i] * scal;
            __syncthreads();
            if (c == 0) {
                double* vb_ = ws.vbuf + (size_t)(k & 1) * P * M + so;
                for (int i = k + 1 + tid; i < M; i += TRD_THREADS) vb_[i] = vn[i];
                if (tid == 0) {
                    ws.d[so + k] = dk;
                    ws.e[so + k] = beta;
                    ws.tau[so + k] = tau;
                }
            }
            // ---- pass over the owned rows below k
            double* pb = ws.pbuf + (size_t)(k & 1) * P * M + so;
            int i0 = k + 1;
            i0 += ((c - i0) % C + C) % C;  // first owned row >= k+1
            for (int i = i0 + C * warp; i < M; i += C * NW) {
                double* row = G + (size_t)i * M;
                const double vi = (k > 0) ? vp[i] : 0.0, wi = (k > 0) ? wp[i] : 0.0;
                double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
                int j = k + 1 + lane;
                for (; j + 96 < M; j += 128) {  // four independent loads per lane in flight
                    double b0 = __ldcg(row + j), b1 = __ldcg(row + j + 32), b2 = __ldcg(row + j + 64), b3 = __ldcg(row + j + 96);
                    if (k > 0) {
                        b0 -= (__dmul_rn(vi, wp[j]) + __dmul_rn(wi, vp[j]));
                        b1 -= (__dmul_rn(vi, wp[j + 32]) + __dmul_rn(wi, vp[j + 32]));
                        b2 -= (__dmul_rn(vi, wp[j + 64]) + __dmul_rn(wi, vp[j + 64]));
                        b3 -= (__dmul_rn(vi, wp[j + 96]) + __dmul_rn(wi, vp[j + 96]));
                        row[j] = b0;
                        row[j + 32] = b1;
                        row[j + 64] = b2;
                        row[j + 96] = b3;
                    }
                    a0 = fma(b0, vn[j], a0);
                    a1 = fma(b1, vn[j + 32], a1);
                    a2 = fma(b2, vn[j + 64], a2);
                    a3 = fma(b3, vn[j + 96], a3);
                }
                for (; j < M; j += 32) {
                    double b0 = __ldcg(row + j);
                    if (k > 0) {
                        b0 -= (__dmul_rn(vi, wp[j]) + __dmul_rn(wi, vp[j]));
                        row[j] = b0;
                    }
                    a0 = fma(b0, vn[j], a0);
                }
                a0 = warp_sum((a0 + a1) + (a2 + a3));
                if (lane == 0) pb[i] = tau * a0;
            }
        }
        if (CLUSTER) cluster_sync_all(); else jw_grid_barrier(bar, phase);
    }
    // last diagonal entry (its pending update was applied by the pass of column M-2)
    for (int vb = blockIdx.x; vb < nv; vb += gridDim.x) {
        const int sl = vb / C, c = vb - sl * C, s = s_off + sl;
        if (c == 0 && tid == 0) {
            ws.d[(size_t)s * M + M - 1] = __ldcg(Gws + (size_t)s * M * M + (size_t)(M - 1) * M + M - 1);
            ws.e[(size_t)s * M + M - 1] = 0.0;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// The same recurrence with the submatrix RESIDENT IN THE DISTRIBUTED SHARED MEMORY of the slice's cluster (small M: the
// BASELINE configs, M = 192-256, and the Table-I-shaped case, M = 416).  CTA c of the C-CTA cluster keeps rows i = c (mod C)
// of B_s in its shared memory for the whole reduction (8 M^2 / C bytes), so the pass over the owned rows is shared-memory
// traffic only; what crosses CTAs is small and goes through DSMEM: every CTA reads row k from its owner's shared memory
// (column k of the symmetric matrix), and the owner of row i stores p_k[i] into every CTA's copy of p.  One hardware cluster
// barrier per column orders those stores; no global-memory round trip is left on the per-column chain (the L2-resident
// version: ~8 us per column of dependent L2 loads, stores and barriers).  Reflectors, tau, d, e still go to global memory
// (CTA 0), where the later kernels expect them.  Bitwise identical to sytrd_kernel: same operations in the same order.
// Dynamic shared memory: Gs[rpc][M], vA[M], vB[M], wp[M], pn[2][M].
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t trd_mapa(uint32_t addr, uint32_t cta) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(cta));
    return r;
}
__device__ __forceinline__ double trd_ld_cluster(uint32_t raddr) {
    double v;
    asm volatile("ld.shared::cluster.f64 %0, [%1];" : "=d"(v) : "r"(raddr) : "memory");
    return v;
}
__device__ __forceinline__ void trd_st_cluster(uint32_t raddr, double v) {
    asm volatile("st.shared::cluster.f64 [%0], %1;" ::"r"(raddr), "d"(v) : "memory");
}

inline size_t sytrd_dsmem_bytes(int M, int C) { return ((size_t)((M + C - 1) / C) * M + 5 * (size_t)M) * sizeof(double); }

__global__ void __launch_bounds__(TRD_THREADS, 1)
sytrd_dsmem_kernel(const double* __restrict__ A, int64_t N, int32_t M, SliceTable tab, double* __restrict__ Gws, TriWs ws,
                   int32_t P, int32_t s_off, int32_t C, int32_t precopied) {
    extern __shared__ double sm[];
    const int rpc = (M + C - 1) / C;  // rows per CTA
    double* Gs = sm;                   // own rows: local row li = i / C
    double* vbuf0 = Gs + (size_t)rpc * M;
    double* vbuf1 = vbuf0 + M;
    double* wp = vbuf1 + M;            // w_{k-1}
    double* pn = wp + M;               // p of the column, [2][M] by column parity; every CTA holds the full vector
    __shared__ double red[TRD_THREADS / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = TRD_THREADS / 32;
    const int c = (int)cluster_ctarank();
    const int s = s_off + blockIdx.x / C;
    const int lo = tab.lo[s];
    const size_t so = (size_t)s * M;
    double* G = Gws + (size_t)s * M * M;  // global copy: receives the reflectors
    const uint32_t Gs_u32 = (uint32_t)__cvta_generic_to_shared(Gs), pn_u32 = (uint32_t)__cvta_generic_to_shared(pn);

    for (int li = warp; li < rpc; li += NW) {  // own rows of B_s (from A, or from the packed blocks pfsm_solve_host uploaded)
        const int i = li * C + c;
        if (i >= M) break;
        const double* a = precopied ? G + (size_t)i * M : A + (size_t)(lo + i) * N + lo;
        for (int j = lane; j < M; j += 32) Gs[(size_t)li * M + j] = a[j];
    }
    for (int i = tid; i < M; i += TRD_THREADS) vbuf0[i] = vbuf1[i] = 0.0;
    cluster_sync_all();

    double tau_p = 0.0;
    for (int k = 0; k <= M - 2; ++k) {
        double* vn = (k & 1) ? vbuf1 : vbuf0;        // v_k
        const double* vp = (k & 1) ? vbuf0 : vbuf1;  // v_{k-1}
        // ---- prologue: row k (= column k of the symmetric matrix) from its owner's shared memory
        double bk[2];  // M <= 1024 = 2 x 512
        {
            const uint32_t rrow = trd_mapa(Gs_u32 + (uint32_t)(((size_t)(k / C) * M) * 8), (uint32_t)(k % C));
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int i = k + tid + TRD_THREADS * e;
                bk[e] = (i < M) ? trd_ld_cluster(rrow + 8u * (uint32_t)i) : 0.0;
            }
        }
        if (k > 0) {
            const double* pv_ = pn + (size_t)((k - 1) & 1) * M;
            double acc = 0.0;
            for (int i = k + tid; i < M; i += TRD_THREADS) {
                const double v = vp[i], p = pv_[i];
                wp[i] = p;
                acc = fma(p, v, acc);
            }
            const double pv = block_sum_512(acc, red);
            const double hf = 0.5 * tau_p * pv;
            for (int i = k + tid; i < M; i += TRD_THREADS) wp[i] = fma(-hf, vp[i], wp[i]);
            __syncthreads();
            if (c == 0)  // row k-1 is dead: keep reflector k-1 there (columns k .., leading 1 included)
                for (int i = k + tid; i < M; i += TRD_THREADS) G[(size_t)(k - 1) * M + i] = vp[i];
        }
        double acc = 0.0;
        {
            const double wk = (k > 0) ? wp[k] : 0.0, vk = (k > 0) ? vp[k] : 0.0;
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int i = k + tid + TRD_THREADS * e;
                if (i < M) {
                    double b = bk[e];
                    if (k > 0) b -= (__dmul_rn(vp[i], wk) + __dmul_rn(wp[i], vk));
                    vn[i] = b;
                    if (i >= k + 2) acc = fma(b, b, acc);
                }
            }
        }
        const double xn2 = block_sum_512(acc, red);  // (its barriers also publish vn)
        const double dk = vn[k], alpha = vn[k + 1];
        double tau = 0.0, beta = alpha, scal = 0.0;
        if (xn2 > 0.0) {
            beta = -copysign(sqrt(fma(alpha, alpha, xn2)), alpha);
            tau = (beta - alpha) / beta;
            scal = 1.0 / (alpha - beta);
        }
        __syncthreads();
        for (int i = k + 1 + tid; i < M; i += TRD_THREADS) vn[i] = (i == k + 1) ? 1.0 : vn[i] * scal;
        __syncthreads();
        if (c == 0 && tid == 0) {
            ws.d[so + k] = dk;
            ws.e[so + k] = beta;
            ws.tau[so + k] = tau;
        }
        // ---- pass over the owned rows below k (shared memory only); p_k[i] goes to every CTA of the cluster
        const uint32_t pdst = pn_u32 + (uint32_t)((size_t)(k & 1) * M * 8);
        int li0 = (k + 1) / C;
        if (li0 * C + c < k + 1) ++li0;  // first owned row >= k+1
        for (int li = li0 + warp; li < rpc; li += NW) {
            const int i = li * C + c;
            if (i >= M) break;
            double* row = Gs + (size_t)li * M;
            const double vi = (k > 0) ? vp[i] : 0.0, wi = (k > 0) ? wp[i] : 0.0;
            double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
            int j = k + 1 + lane;
            for (; j + 96 < M; j += 128) {
                double b0 = row[j], b1 = row[j + 32], b2 = row[j + 64], b3 = row[j + 96];
                if (k > 0) {
                    b0 -= (__dmul_rn(vi, wp[j]) + __dmul_rn(wi, vp[j]));
                    b1 -= (__dmul_rn(vi, wp[j + 32]) + __dmul_rn(wi, vp[j + 32]));
                    b2 -= (__dmul_rn(vi, wp[j + 64]) + __dmul_rn(wi, vp[j + 64]));
                    b3 -= (__dmul_rn(vi, wp[j + 96]) + __dmul_rn(wi, vp[j + 96]));
                    row[j] = b0;
                    row[j + 32] = b1;
                    row[j + 64] = b2;
                    row[j + 96] = b3;
                }
                a0 = fma(b0, vn[j], a0);
                a1 = fma(b1, vn[j + 32], a1);
                a2 = fma(b2, vn[j + 64], a2);
                a3 = fma(b3, vn[j + 96], a3);
            }
            for (; j < M; j += 32) {
                double b0 = row[j];
                if (k > 0) {
                    b0 -= (__dmul_rn(vi, wp[j]) + __dmul_rn(wi, vp[j]));
                    row[j] = b0;
                }
                a0 = fma(b0, vn[j], a0);
            }
            a0 = warp_sum((a0 + a1) + (a2 + a3));
            if (lane < C) trd_st_cluster(trd_mapa(pdst + 8u * (uint32_t)i, (uint32_t)lane), tau * a0);
        }
        tau_p = tau;
        cluster_sync_all();
    }
    // last diagonal entry (its pending update was applied by the pass of column M-2)
    if (tid == 0 && (M - 1) % C == c) {
        ws.d[so + M - 1] = Gs[(size_t)((M - 1) / C) * M + M - 1];
        ws.e[so + M - 1] = 0.0;
    }
}

// ---------------------------------------------------------------------------------------------
// The same recurrence on the LOWER TRIANGLE only (entries j <= i): half the memory traffic, 8 (M-k)^2 bytes per column.
// The product p = B v needs, for row i, the row part sum_{j<=i} B[i][j] v[j] and the column part sum_{r>i} B[r][i] v[r].
// The active triangle is cut into 32 x 32 tiles (row block Rb, column strip S <= Rb), dealt cyclically to the warps of
// the slice's CTAs.  A warp walks the 32 rows of its tile with lane = column: the column part accumulates in a register,
// the row part is a shuffle reduction per row.  Tiles write their partial sums to rowbuf[S][i] and colbuf[Rb][j] (each
// entry written by exactly one warp), a grid barrier follows, then p[i] = tau (sum_S rowbuf[S][i] + sum_Rb colbuf[Rb][i])
// is summed in fixed order by the CTA that owns a contiguous range of rows, and a second grid barrier publishes p.
// No atomics: bitwise reproducible.  Column k itself (B[i][k], i > k) is read with stride M in the prologue.
// Reflector k goes to the (unused) upper part of row k: columns k+1 .., leading 1 stored.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(TRD_THREADS, 1)
sytrd_half_kernel(const double* __restrict__ A, int64_t N, int32_t M, SliceTable tab, double* __restrict__ Gws, TriWs ws,
                  int32_t P, int32_t s_off, int32_t ns, int32_t C, unsigned int* __restrict__ bar, int32_t precopied) {
    extern __shared__ double sm[];
    double* vp = sm;          // v_{k-1}
    double* wp = sm + M;      // w_{k-1}
    double* vn = sm + 2 * M;  // v_k
    __shared__ double red[TRD_THREADS / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = TRD_THREADS / 32;
    unsigned int phase = 0;
    const int nv = ns * C;
    const int nb = (M + 31) / 32;
    const size_t bufs = (size_t)nb * M;  // rowbuf / colbuf doubles per slice

    for (int vb = blockIdx.x; vb < nv && !precopied; vb += gridDim.x) {
        const int sl = vb / C, c = vb - sl * C, s = s_off + sl;
        const int lo = tab.lo[s];
        double* G = Gws + (size_t)s * M * M;
        for (int i = c + C * warp; i < M; i += C * NW) {
            const double* a = A + (size_t)(lo + i) * N + lo;
            for (int j = lane; j <= i; j += 32) G[(size_t)i * M + j] = a[j];
        }
    }
    jw_grid_barrier(bar, phase);

    for (int k = 0; k <= M - 2; ++k) {
        const int b0 = (k + 1) / 32, nbk = nb - b0, ntiles = nbk * (nbk + 1) / 2;
        for (int vb = blockIdx.x; vb < nv; vb += gridDim.x) {
            const int sl = vb / C, c = vb - sl * C, s = s_off + sl;
            double* G = Gws + (size_t)s * M * M;
            const size_t so = (size_t)s * M;
            __syncthreads();
            // ---- prologue (as in sytrd_kernel; column k is read down the column)
            if (k > 0) {
                const double tau_p = __ldcg(ws.tau + so + k - 1);
                const double* pv_ = ws.pbuf + (size_t)((k - 1) & 1) * P * M + so;
                const double* vv_ = ws.vbuf + (size_t)((k - 1) & 1) * P * M + so;
                double acc = 0.0;
                for (int i = k + tid; i < M; i += TRD_THREADS) {
                    const double v = __ldcg(vv_ + i), p = __ldcg(pv_ + i);
                    vp[i] = v;
                    wp[i] = p;
                    acc = fma(p, v, acc);
                }
                const double pv = block_sum_512(acc, red);
                const double hf = 0.5 * tau_p * pv;
                for (int i = k + tid; i < M; i += TRD_THREADS) wp[i] = fma(-hf, vp[i], wp[i]);
                __syncthreads();
            }
            double acc = 0.0;
            {
                const double wk = (k > 0) ? wp[k] : 0.0, vk = (k > 0) ? vp[k] : 0.0;
                for (int i = k + tid; i < M; i += TRD_THREADS) {
                    // column k: written contiguously by the previous pass (k = 0: down the column of the copy)
                    double b = (k > 0) ? __ldcg(ws.colk + (size_t)((k - 1) & 1) * P * M + so + i) : __ldcg(G + (size_t)i * M);
                    if (k > 0) b -= (__dmul_rn(vp[i], wk) + __dmul_rn(wp[i], vk));
                    vn[i] = b;
                    if (i >= k + 2) acc = fma(b, b, acc);
                }
            }
            const double xn2 = block_sum_512(acc, red);
            const double dk = vn[k], alpha = vn[k + 1];
            double tau = 0.0, beta = alpha, scal = 0.0;
            if (xn2 > 0.0) {
                beta = -copysign(sqrt(fma(alpha, alpha, xn2)), alpha);
                tau = (beta - alpha) / beta;
                scal = 1.0 / (alpha - beta);
            }
            __syncthreads();
            for (int i = k + 1 + tid; i < M; i += TRD_THREADS) vn[i] = (i == k + 1) ? 1.0 : vn[i] * scal;
            __syncthreads();
            if (c == 0) {
                double* vb_ = ws.vbuf + (size_t)(k & 1) * P * M + so;
                for (int i = k + 1 + tid; i < M; i += TRD_THREADS) {
                    vb_[i] = vn[i];
                    G[(size_t)k * M + i] = vn[i];  // reflector k: upper part of row k, never touched by the recurrence
                }
                if (tid == 0) {
                    ws.d[so + k] = dk;
                    ws.e[so + k] = beta;
                    ws.tau[so + k] = tau;
                }
            }
            // ---- pass over the tiles of the active lower triangle
            double* rowbuf = ws.rowbuf + (size_t)s * bufs;
            double* colbuf = ws.colbuf + (size_t)s * bufs;
            double* nextcol = ws.colk + (size_t)(k & 1) * P * M + so;
            for (int t = c * NW + warp; t < ntiles; t += C * NW) {
                int rb = (int)((sqrt(8.0 * (double)t + 1.0) - 1.0) * 0.5);
                while ((rb + 1) * (rb + 2) / 2 <= t) ++rb;
                while (rb * (rb + 1) / 2 > t) --rb;
                const int S = b0 + (t - rb * (rb + 1) / 2), Rb = b0 + rb;
                const int j = 32 * S + lane, ib = 32 * Rb;
                const bool jok = j >= k + 1 && j < M;
                const double wj = (jok && k > 0) ? wp[j] : 0.0, vj = (jok && k > 0) ? vp[j] : 0.0, vnj = jok ? vn[j] : 0.0;
                double colacc = 0.0;
                double b[32];
#pragma unroll
                for (int r = 0; r < 32; ++r) {  // the whole tile column of this lane in flight at once
                    const int i = ib + r;
                    b[r] = (jok && i < M && j <= i) ? __ldcg(G + (size_t)i * M + j) : 0.0;
                }
#pragma unroll
                for (int r = 0; r < 32; ++r) {
                    const int i = ib + r;
                    const bool ok = jok && i < M && j <= i;  // (i >= k+1 follows from j >= k+1)
                    double bb = b[r];
                    if (k > 0 && ok) {
                        bb -= (__dmul_rn(vp[i], wj) + __dmul_rn(wp[i], vj));
                        G[(size_t)i * M + j] = bb;
                    }
                    if (ok && j == k + 1) nextcol[i] = bb;  // column k+1 for the next prologue (update k still pending)
                    if (ok && j < i) colacc = fma(bb, vn[i], colacc);
                    b[r] = bb * vnj;
                }
                // row sums: transposed butterfly, 31 shuffles; lane l ends with the sum of row ib + l over the 32 columns
#pragma unroll
                for (int h = 16; h >= 1; h >>= 1) {
                    const bool up = (lane & h) != 0;
#pragma unroll
                    for (int r = 0; r < h; ++r) {
                        const double send = up ? b[r] : b[r + h], keep = up ? b[r + h] : b[r];
                        b[r] = keep + __shfl_xor_sync(0xffffffffu, send, h);
                    }
                }
                const double myrow = b[0];
                const int i = ib + lane;
                if (i >= k + 1 && i < M) rowbuf[(size_t)S * M + i] = myrow;
                if (j < M) colbuf[(size_t)Rb * M + j] = colacc;
            }
        }
        jw_grid_barrier(bar, phase);
        // ---- p = tau (row parts + column parts), contiguous row ranges per CTA, thread per row, fixed order
        for (int vb = blockIdx.x; vb < nv; vb += gridDim.x) {
            const int sl = vb / C, c = vb - sl * C, s = s_off + sl;
            const size_t so = (size_t)s * M;
            const double tau = __ldcg(ws.tau + so + k);
            const double* rowbuf = ws.rowbuf + (size_t)s * bufs;
            const double* colbuf = ws.colbuf + (size_t)s * bufs;
            double* pb = ws.pbuf + (size_t)(k & 1) * P * M + so;
            const int L = M - k - 1, per = (L + C - 1) / C;
            const int i0 = k + 1 + c * per, i1 = min(M, i0 + per);
            // two threads per row (even / odd terms), 8 loads in flight each; terms in fixed order: strips b0 .. bi of
            // rowbuf, then row blocks bi .. nb-1 of colbuf; the two partial sums are added by a shuffle (commutative: same bits)
            for (int base = 0; base < per; base += TRD_THREADS / 2) {
                const int i = i0 + base + (tid >> 1), sub = tid & 1;
                const bool valid = i < i1;
                const int bi = i / 32;
                const int n1 = bi - b0 + 1, nt = valid ? n1 + nb - bi : 0;
                double a = 0.0;
                for (int q0 = sub; q0 < nt; q0 += 16) {
                    double x[8];
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        const int q = q0 + 2 * u;
                        x[u] = (q >= nt) ? 0.0
                               : (q < n1) ? __ldcg(rowbuf + (size_t)(b0 + q) * M + i)
                                          : __ldcg(colbuf + (size_t)(bi + q - n1) * M + i);
                    }
#pragma unroll
                    for (int u = 0; u < 8; ++u) a += x[u];
                }
                a += __shfl_xor_sync(0xffffffffu, a, 1);
                if (valid && sub == 0) pb[i] = tau * a;
            }
        }
        jw_grid_barrier(bar, phase);
    }
    for (int vb = blockIdx.x; vb < nv; vb += gridDim.x) {
        const int sl = vb / C, c = vb - sl * C, s = s_off + sl;
        if (c == 0 && tid == 0) {
            ws.d[(size_t)s * M + M - 1] = __ldcg(Gws + (size_t)s * M * M + (size_t)(M - 1) * M + M - 1);
            ws.e[(size_t)s * M + M - 1] = 0.0;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Eigenvalue of local rank off + t of T_s by bisection.  count(x) = number of eigenvalues < x = number of sign changes
// of the Sturm sequence p_i = (d_i - x) p_{i-1} - e_{i-1}^2 p_{i-2}, p_{-1} = 1 (= negative pivots of LDL^T).
// grid.x = ceil(mmax / (TRI_THREADS / 32)) (a warp per eigenvalue), grid.y = ns.  Dynamic shared memory: d[M], e2[M].
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(TRI_THREADS)
tri_bisect_kernel(int32_t M, SliceTable tab, TriWs ws, int32_t s_off) {
    extern __shared__ double sm[];
    double* d = sm;
    double* e2 = sm + M;
    __shared__ double rlo[TRI_THREADS / 32], rhi[TRI_THREADS / 32], rem[TRI_THREADS / 32];
    const int s = s_off + blockIdx.y, tid = threadIdx.x;
    const size_t so = (size_t)s * M;
    double glo = 1e300, ghi = -1e300, emax = 0.0;
    for (int i = tid; i < M; i += TRI_THREADS) {
        const double di = ws.d[so + i], ei = (i < M - 1) ? ws.e[so + i] : 0.0, em = (i > 0) ? ws.e[so + i - 1] : 0.0;
        d[i] = di;
        e2[i] = ei * ei;
        const double r = fabs(ei) + fabs(em);
        glo = fmin(glo, di - r);
        ghi = fmax(ghi, di + r);
        emax = fmax(emax, ei * ei);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        glo = fmin(glo, __shfl_xor_sync(0xffffffffu, glo, o));
        ghi = fmax(ghi, __shfl_xor_sync(0xffffffffu, ghi, o));
        emax = fmax(emax, __shfl_xor_sync(0xffffffffu, emax, o));
    }
    if ((tid & 31) == 0) {
        rlo[tid >> 5] = glo;
        rhi[tid >> 5] = ghi;
        rem[tid >> 5] = emax;
    }
    __syncthreads();
    for (int w = 0; w < TRI_THREADS / 32; ++w) {
        glo = fmin(glo, rlo[w]);
        ghi = fmax(ghi, rhi[w]);
        emax = fmax(emax, rem[w]);
    }
    // One WARP per eigenvalue: 32 probes x_l = lo + (l + 1)(hi - lo)/33 per round (multi-section), so an interval shrinks
    // 33-fold per serial Sturm chain instead of 2-fold: ~11 rounds instead of ~55.
    const int lane = tid & 31;
    const int t = blockIdx.x * (TRI_THREADS / 32) + (tid >> 5);
    if (t >= tab.cnt[s]) return;
    const int rank = tab.off[s] + t;
    const double pivmin = 2.2250738585072014e-308 * fmax(1.0, emax);
    const double span = fmax(fabs(glo), fabs(ghi));
    double lo = glo - 2.0 * 2.220446049250313e-16 * span * M - 2.0 * pivmin;
    double hi = ghi + 2.0 * 2.220446049250313e-16 * span * M + 2.0 * pivmin;
    for (int it = 0; it < 64; ++it) {
        if (hi - lo <= 2.220446049250313e-16 * (fmax(fabs(lo), fabs(hi)) + 0.125 * span) + 2.0 * pivmin) break;
        const double hstep = (hi - lo) * (1.0 / 33.0);
        const double mid = fma((double)(lane + 1), hstep, lo);
        // Sturm sequence in product form p_i = (d_i - x) p_{i-1} - e_{i-1}^2 p_{i-2} (two dependent FMAs per row instead
        // of a division); a sign change between consecutive members = one eigenvalue below x; an exact zero takes the
        // sign opposite to its predecessor; both members are rescaled every four rows against over/underflow
        double p0 = 1.0, p1 = d[0] - mid;
        if (p1 == 0.0) p1 = -pivmin;
        unsigned int cnt = p1 < 0.0 ? 1u : 0u;
        auto step = [&](int i) {
            double p2 = fma(d[i] - mid, p1, -e2[i - 1] * p0);
            if (p2 == 0.0) p2 = -copysign(fmax(fabs(p1), 1e-280) * 1e-20, p1);
            cnt += ((unsigned int)(__double2hiint(p2) ^ __double2hiint(p1))) >> 31;  // sign change
            p0 = p1;
            p1 = p2;
        };
        int i = 1;
        for (; i + 3 < M; i += 4) {
            step(i);
            step(i + 1);
            step(i + 2);
            step(i + 3);
            const double a = fmax(fabs(p0), fabs(p1));
            if (a > 1e120) {
                p0 *= 1e-120;
                p1 *= 1e-120;
            } else if (a < 1e-120) {
                p0 *= 1e120;
                p1 *= 1e120;
            }
        }
        for (; i < M; ++i) step(i);
        // first probe with more than `rank` eigenvalues below it bounds the eigenvalue from above, its left neighbour
        // (or the old lo) from below
        const unsigned above = __ballot_sync(0xffffffffu, (int)cnt > rank);
        const int f = above ? __ffs(above) - 1 : 32;
        const double nhi = __shfl_sync(0xffffffffu, mid, f & 31), nlo = __shfl_sync(0xffffffffu, mid, (f + 31) & 31);
        const double olo = lo, ohi = hi;
        hi = (f < 32) ? nhi : ohi;
        lo = (f > 0) ? nlo : olo;
        if (!(hi > lo) || (lo == olo && hi == ohi)) break;  // no representable progress
    }
    if (lane == 0) ws.lam[tab.g0[s] + t] = 0.5 * (lo + hi);
}

// counter-based uniform in (-1, 1): splitmix64 finalizer of (vector, row)
__device__ __forceinline__ double tri_start_value(uint32_t vec, uint32_t row) {
    uint64_t z = ((uint64_t)vec << 32 | row) * 0x9E3779B97F4A7C15ull + 0xD1B54A32D192ED03ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    z ^= z >> 31;
    return ((double)(z >> 11) + 0.5) * (2.0 / 9007199254740992.0) - 1.0;
}

// ---------------------------------------------------------------------------------------------
// Eigenvector of T_s for eigenvalue lam[g0 + t]: inverse iteration (the LAPACK dstein scheme without its cluster
// re-orthogonalization).  T - x I = P L U with partial pivoting (the dgttrf recurrence), pivots below eps ||T|| are
// replaced by eps ||T||; three solves from a random start, the vector rescaled to unit 2-norm between solves.
// Factors and vector live in global memory as [row i][vector g], g = g0 + t: a warp touches 32 consecutive doubles.
// Output: z in ws.f[4] (not normalized), ws.zscale[g] = 1 / ||z||_2.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(TRI_THREADS)
tri_invit_kernel(int64_t N, int32_t M, SliceTable tab, TriWs ws, int32_t s_off, unsigned long long* info) {
    extern __shared__ double sm[];
    double* d = sm;
    double* e = sm + M;
    __shared__ double rmx[TRI_THREADS / 32];
    const int s = s_off + blockIdx.y, tid = threadIdx.x;
    const size_t so = (size_t)s * M;
    double tmax = 0.0;
    for (int i = tid; i < M; i += TRI_THREADS) {
        const double di = ws.d[so + i], ei = (i < M - 1) ? ws.e[so + i] : 0.0;
        d[i] = di;
        e[i] = ei;
        tmax = fmax(tmax, fabs(di) + 2.0 * fabs(ei));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) tmax = fmax(tmax, __shfl_xor_sync(0xffffffffu, tmax, o));
    if ((tid & 31) == 0) rmx[tid >> 5] = tmax;
    __syncthreads();
    for (int w = 0; w < TRI_THREADS / 32; ++w) tmax = fmax(tmax, rmx[w]);
    const int t = blockIdx.x * TRI_THREADS + tid;
    const int m = tab.cnt[s];
    if (t >= m) return;
    const int g0 = tab.g0[s];
    const size_t g = (size_t)g0 + t;
    const double EPS = 2.220446049250313e-16;
    // shifts of eigenvalues closer than 10 eps |lambda| are pushed apart (dstein); the chain is followed from the
    // slice's first eigenvalue so that every thread derives the same perturbed sequence
    double x = ws.lam[g0];
    for (int j = 1; j <= t; ++j) {
        const double xj = ws.lam[g0 + j];
        const double pertol = 10.0 * EPS * fmax(fabs(xj), 1e-3 * tmax);  // (floor: eigenvalues clustered at zero are pushed apart too)
        x = (xj - x < pertol) ? x + pertol : xj;
    }
    const double pivtol = fmax(EPS * tmax, 1e-300);
    double* uinv = ws.f[0] + g;  // 1 / U[i][i]
    double* u1 = ws.f[1] + g;    // U[i][i+1]
    double* u2 = ws.f[2] + g;    // U[i][i+2]
    double* lm = ws.f[3] + g;    // multiplier of elimination step i
    double* z = ws.f[4] + g;
    unsigned char* pv = ws.piv + g;
    const size_t st = (size_t)N;
    {
        double cur_d = d[0] - x, cur_du = (M > 1) ? e[0] : 0.0;
        for (int i = 0; i < M - 1; ++i) {
            const double sub = e[i], nxt_d = d[i + 1] - x, nxt_du = (i + 1 < M - 1) ? e[i + 1] : 0.0;
            if (fabs(cur_d) >= fabs(sub)) {
                double piv = cur_d;
                if (fabs(piv) < pivtol) piv = (piv < 0.0) ? -pivtol : pivtol;
                const double inv = 1.0 / piv;
                const double f = sub * inv;
                uinv[i * st] = inv;
                u1[i * st] = cur_du;
                u2[i * st] = 0.0;
                lm[i * st] = f;
                pv[i * st] = 0;
                cur_d = fma(-f, cur_du, nxt_d);
                cur_du = nxt_du;
            } else {
                const double inv = 1.0 / sub;
                const double f = cur_d * inv;
                uinv[i * st] = inv;
                u1[i * st] = nxt_d;
                u2[i * st] = nxt_du;
                lm[i * st] = f;
                pv[i * st] = 1;
                cur_d = fma(-f, nxt_d, cur_du);
                cur_du = -f * nxt_du;
            }
        }
        double piv = cur_d;
        if (fabs(piv) < pivtol) piv = (piv < 0.0) ? -pivtol : pivtol;
        uinv[(size_t)(M - 1) * st] = 1.0 / piv;
    }
    double scale = 1.0;
    for (int iter = 0; iter < 3; ++iter) {
        // forward: L^-1 P^T b   (b = scale * previous z, or the random start)
        // (operands of IB rows are requested together: the recurrences are short, the global-memory latency is not)
        constexpr int IB = 8;
        double bi = (iter == 0) ? tri_start_value((uint32_t)g, 0u) : z[0] * scale;
        for (int i0 = 0; i0 < M - 1; i0 += IB) {
            double bnv[IB], fv[IB];
            unsigned char pvv[IB];
#pragma unroll
            for (int u = 0; u < IB; ++u) {
                const int i = i0 + u;
                if (i < M - 1) {
                    bnv[u] = (iter == 0) ? tri_start_value((uint32_t)g, (uint32_t)(i + 1)) : z[(size_t)(i + 1) * st] * scale;
                    fv[u] = lm[i * st];
                    pvv[u] = pv[i * st];
                }
            }
#pragma unroll
            for (int u = 0; u < IB; ++u) {
                const int i = i0 + u;
                if (i < M - 1) {
                    if (pvv[u]) {
                        z[i * st] = bnv[u];
                        bi = fma(-fv[u], bnv[u], bi);
                    } else {
                        z[i * st] = bi;
                        bi = fma(-fv[u], bi, bnv[u]);
                    }
                }
            }
        }
        // backward: U^-1
        double x1 = bi * uinv[(size_t)(M - 1) * st], x2 = 0.0;
        z[(size_t)(M - 1) * st] = x1;
        double ss = x1 * x1;
        for (int i0 = M - 2; i0 >= 0; i0 -= IB) {
            double zv[IB], a1[IB], a2[IB], iv[IB];
#pragma unroll
            for (int u = 0; u < IB; ++u) {
                const int i = i0 - u;
                if (i >= 0) {
                    zv[u] = z[i * st];
                    a1[u] = u1[i * st];
                    a2[u] = u2[i * st];
                    iv[u] = uinv[i * st];
                }
            }
#pragma unroll
            for (int u = 0; u < IB; ++u) {
                const int i = i0 - u;
                if (i >= 0) {
                    const double xi = (zv[u] - a1[u] * x1 - a2[u] * x2) * iv[u];
                    z[i * st] = xi;
                    ss = fma(xi, xi, ss);
                    x2 = x1;
                    x1 = xi;
                }
            }
        }
        scale = rsqrt(ss);
        // guard against overflow of the sum of squares (growth ~ 1/(eps ||T||) per solve from a unit vector)
        if (!(ss < 1e300)) {
            double mx = 0.0;
            for (int i = 0; i < M; ++i) mx = fmax(mx, fabs(z[i * st]));
            double s2 = 0.0;
            for (int i = 0; i < M; ++i) {
                const double q = z[i * st] / mx;
                s2 = fma(q, q, s2);
            }
            scale = 1.0 / (mx * sqrt(s2));
        }
    }
    ws.zscale[g] = scale;
    // convergence: the last solve (T - x I) z' = z, ||z|| = 1, must have grown the vector to ||z'|| >= 1 / (sqrt(eps) ||T||),
    // i.e. left a residual <= sqrt(eps) ||T|| (one more solve squares it); else the slice is flagged as the Jacobi kernels do
    if (!(scale <= 1.4901161193847656e-08 * tmax) && tmax > 0.0) atomicMin(info, (unsigned long long)(N + s + 1));
}

// ---------------------------------------------------------------------------------------------
// Eigenvalue clusters (LAPACK dstein's re-orthogonalization, restricted to the gaps that need it).  Inverse iteration
// without it delivers the vectors of a pair with gap g to eps ||T|| / g; for g below TRI_CLUSTER_TOL ||T|| two vectors can
// come out numerically parallel, and step 4 would then orthonormalize noise.  For every run of consecutive eigenvalues
// closer than that, members 2, 3, .. are -- one after the other -- orthogonalized against the earlier members (modified
// Gram-Schmidt), normalized and put through one more inverse-iteration solve with their own stored LU factors, three
// times, ending on an orthogonalization.  Runs are independent: the CX CTAs of a slice (grid.x) take them round-robin;
// inside a run the members follow each other on one CTA.  The dot products run over the CTA (fixed order); the solve is
// the serial recurrence on one thread, from SHARED memory (STAGED: the vector and its LU factors are staged there once
// per member, 41 M bytes; the global-memory version pays an L2 round trip per row and is kept for M > 4096).  Exactly
// degenerate spectra (the paper's diamond cell is "highly degenerate") put every vector through this pass:
// step 2 of a 13-fold degenerate 256 x 256 matrix took 24 ms with one CTA per slice and global-memory solves, against 1.3 ms
// for a generic spectrum.
// Dynamic shared memory: lam[mmax] doubles; STAGED: + z, 1/U_ii, U_i,i+1, U_i,i+2, L multipliers [M] doubles, pivots [M] bytes.
// ---------------------------------------------------------------------------------------------
constexpr double TRI_CLUSTER_TOL = 1e-7;
constexpr int TRC_THREADS = 256;
constexpr int TRC_STAGED_MAX_M = 4096;

constexpr int TRC_CHUNK = 1024;  // rows per staging chunk of the solve when M > TRC_STAGED_MAX_M

inline size_t tri_cluster_smem_bytes(int M, int mmax, bool staged) {
    return (size_t)mmax * 8 + (size_t)(staged ? M : TRC_CHUNK) * 41 + 16;
}

__device__ __forceinline__ double trc_block_sum(double v, double* red) {
    v = warp_sum(v);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < TRC_THREADS / 32; ++w) t += red[w];
    return t;
}

template <bool STAGED>
__global__ void __launch_bounds__(TRC_THREADS)
tri_cluster_kernel(int64_t N, int32_t M, SliceTable tab, TriWs ws, int32_t s_off, int32_t mmax) {
    extern __shared__ double trc_sm[];
    double* lam_s = trc_sm;                          // the slice's eigenvalues
    const int SL = STAGED ? M : TRC_CHUNK;           // rows the staging arrays hold
    double* zs = trc_sm + mmax;                      // STAGED: the member's vector and LU factors; else one chunk of them
    double* f0 = zs + SL;
    double* f1 = f0 + SL;
    double* f2 = f1 + SL;
    double* f3 = f2 + SL;
    unsigned char* pvs = reinterpret_cast<unsigned char*>(f3 + SL);
    __shared__ double red[TRC_THREADS / 32];
    const int s = s_off + blockIdx.y, tid = threadIdx.x;
    const int cta = blockIdx.x, CX = gridDim.x;
    const size_t so = (size_t)s * M;
    const int m = tab.cnt[s], g0 = tab.g0[s];
    double tmax = 0.0;
    for (int i = tid; i < M; i += TRC_THREADS) {
        const double ei = (i < M - 1) ? ws.e[so + i] : 0.0;
        tmax = fmax(tmax, fabs(ws.d[so + i]) + 2.0 * fabs(ei));
    }
    for (int t = tid; t < m; t += TRC_THREADS) lam_s[t] = ws.lam[g0 + t];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) tmax = fmax(tmax, __shfl_xor_sync(0xffffffffu, tmax, o));
    __syncthreads();
    if ((tid & 31) == 0) red[tid >> 5] = tmax;
    __syncthreads();
    for (int w = 0; w < TRC_THREADS / 32; ++w) tmax = fmax(tmax, red[w]);
    const double gaptol = TRI_CLUSTER_TOL * tmax;
    const size_t st = (size_t)N;
    int start = 0;   // first member of the current run
    int runid = -1;  // index of the current run among the runs with at least two members
    // every thread walks the (shared-memory) eigenvalue list the same way: all branches below are block-uniform
    for (int t = 1; t < m; ++t) {
        if (lam_s[t] - lam_s[t - 1] > gaptol) {
            start = t;
            continue;
        }
        if (t == start + 1) ++runid;
        if (runid % CX != cta) continue;
        // eigenvalue t belongs to the run [start, t]: orthogonalize its vector against members start .. t-1
        const size_t g = (size_t)g0 + t;
        double* zg = ws.f[4] + g;
        if (STAGED) {
            for (int i = tid; i < M; i += TRC_THREADS) {
                zs[i] = zg[i * st];
                f0[i] = ws.f[0][g + i * st];
                f1[i] = ws.f[1][g + i * st];
                f2[i] = ws.f[2][g + i * st];
                f3[i] = ws.f[3][g + i * st];
                pvs[i] = ws.piv[g + i * st];
            }
            __syncthreads();
        }
        auto Z = [&](int i) -> double& { return STAGED ? zs[i] : zg[i * st]; };
        for (int it = 0; it < 3; ++it) {
            for (int b = start; b < t; ++b) {
                const double* zb = ws.f[4] + g0 + b;
                const double sb_ = ws.zscale[g0 + b];
                double acc = 0.0;
                for (int i = tid; i < M; i += TRC_THREADS) acc = fma(Z(i), zb[i * st] * sb_, acc);
                const double dot = trc_block_sum(acc, red);
                for (int i = tid; i < M; i += TRC_THREADS) Z(i) = fma(-dot, zb[i * st] * sb_, Z(i));
                __syncthreads();
            }
            double mx = 0.0;  // scaled 2-norm (the vector carries the growth of the solves)
            for (int i = tid; i < M; i += TRC_THREADS) mx = fmax(mx, fabs(Z(i)));
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
            __syncthreads();
            if ((tid & 31) == 0) red[tid >> 5] = mx;
            __syncthreads();
            for (int w = 0; w < TRC_THREADS / 32; ++w) mx = fmax(mx, red[w]);
            const double inv = (mx > 0.0) ? 1.0 / mx : 1.0;
            double acc = 0.0;
            for (int i = tid; i < M; i += TRC_THREADS) {
                const double q = Z(i) * inv;
                acc = fma(q, q, acc);
            }
            const double nrm = sqrt(trc_block_sum(acc, red));
            const double sc = (nrm > 0.0) ? inv / nrm : 1.0;
            for (int i = tid; i < M; i += TRC_THREADS) Z(i) *= sc;
            __syncthreads();
            if (it == 2) break;
            // one more solve with this vector's own factors (the tri_invit_kernel recurrences), by thread 0 from shared memory
            if (STAGED) {
                if (tid == 0) {
                    double bi = zs[0];
                    for (int i = 0; i < M - 1; ++i) {
                        const double bn = zs[i + 1], f = f3[i];
                        if (pvs[i]) {
                            zs[i] = bn;
                            bi = fma(-f, bn, bi);
                        } else {
                            zs[i] = bi;
                            bi = fma(-f, bi, bn);
                        }
                    }
                    double x1 = bi * f0[M - 1], x2 = 0.0;
                    zs[M - 1] = x1;
                    for (int i = M - 2; i >= 0; --i) {
                        const double xi = (zs[i] - f1[i] * x1 - f2[i] * x2) * f0[i];
                        zs[i] = xi;
                        x2 = x1;
                        x1 = xi;
                    }
                }
            } else {
                // M > TRC_STAGED_MAX_M: the vector stays in global memory; the solve walks it in chunks of TRC_CHUNK rows
                // that all threads stage in (operands) and out (results), so that the recurrence never waits on global memory
                const double* uinv = ws.f[0] + g;
                const double* u1 = ws.f[1] + g;
                const double* u2 = ws.f[2] + g;
                const double* lm = ws.f[3] + g;
                const unsigned char* pv = ws.piv + g;
                double bi = zg[0], x1 = 0.0, x2 = 0.0;  // (thread 0's copies carry the recurrences across chunks)
                for (int i0 = 0; i0 < M - 1; i0 += TRC_CHUNK) {  // forward: L^-1 P^T
                    const int n = min(TRC_CHUNK, M - 1 - i0);
                    for (int j = tid; j < n; j += TRC_THREADS) {
                        f0[j] = zg[(size_t)(i0 + j + 1) * st];
                        f3[j] = lm[(size_t)(i0 + j) * st];
                        pvs[j] = pv[(size_t)(i0 + j) * st];
                    }
                    __syncthreads();
                    if (tid == 0) {
                        for (int j = 0; j < n; ++j) {
                            const double bn = f0[j], f = f3[j];
                            if (pvs[j]) {
                                zs[j] = bn;
                                bi = fma(-f, bn, bi);
                            } else {
                                zs[j] = bi;
                                bi = fma(-f, bi, bn);
                            }
                        }
                    }
                    __syncthreads();
                    for (int j = tid; j < n; j += TRC_THREADS) zg[(size_t)(i0 + j) * st] = zs[j];
                    __syncthreads();
                }
                if (tid == 0) {
                    x1 = bi * uinv[(size_t)(M - 1) * st];
                    zg[(size_t)(M - 1) * st] = x1;
                }
                for (int i1 = M - 2; i1 >= 0; i1 -= TRC_CHUNK) {  // backward: U^-1, rows i1, i1 - 1, ..
                    const int n = min(TRC_CHUNK, i1 + 1);
                    for (int j = tid; j < n; j += TRC_THREADS) {
                        const size_t i = (size_t)(i1 - j);
                        f3[j] = zg[i * st];
                        f0[j] = uinv[i * st];
                        f1[j] = u1[i * st];
                        f2[j] = u2[i * st];
                    }
                    __syncthreads();
                    if (tid == 0) {
                        for (int j = 0; j < n; ++j) {
                            const double xi = (f3[j] - f1[j] * x1 - f2[j] * x2) * f0[j];
                            zs[j] = xi;
                            x2 = x1;
                            x1 = xi;
                        }
                    }
                    __syncthreads();
                    for (int j = tid; j < n; j += TRC_THREADS) zg[(size_t)(i1 - j) * st] = zs[j];
                    __syncthreads();
                }
            }
            __syncthreads();
        }
        if (STAGED) {
            for (int i = tid; i < M; i += TRC_THREADS) zg[i * st] = zs[i];
        }
        if (tid == 0) ws.zscale[g] = 1.0;
        __threadfence();  // the next member of the run (same CTA) reads this vector from global memory
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------------
// y = Q z = H_0 H_1 ... H_{M-3} z,  H_k = I - tau_k v_k v_k^T, v_k in row k of the slice's matrix (columns k+1 ..).
// A CTA of 256 threads takes NV eigenvectors and keeps them in REGISTERS: thread t holds rows t + 256 e (e < EPT,
// M <= 256 EPT) of all NV vectors.  Per reflector: v_k is read once per CTA (coalesced, prefetched one reflector
// ahead; rows <= k read as 0 so no predicates are needed), NV dot products are reduced by shuffles and one block
// barrier (partials double-buffered by reflector parity), then the NV axpys.  FP64 FMA issue bound; the reflectors
// (4 M^2 bytes per slice) come from L2.  Writes V[g0 + j][lo .. lo + M) and eps[g0 + j].
// grid.x = ceil(mmax / NV), grid.y = ns.
// ---------------------------------------------------------------------------------------------
constexpr int BT_THREADS = 256;

template <int EPT, int NV>  // NV = 8, 4 or 2; BT_THREADS = 256 (8 warps) is assumed by the cross-warp sum
__global__ void __launch_bounds__(BT_THREADS, 1)
tri_backtransform_kernel(int64_t N, int32_t M, SliceTable tab, const double* __restrict__ Gws, TriWs ws,
                         double* __restrict__ V, double* __restrict__ eps, int32_t s_off) {
    __shared__ double part[2][BT_THREADS / 32][NV];
    const int s = s_off + blockIdx.y, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int t0 = blockIdx.x * NV, cnt = tab.cnt[s];
    if (t0 >= cnt) return;
    const int g0 = tab.g0[s], lo = tab.lo[s];
    const size_t g = (size_t)g0 + t0;
    double x[NV][EPT];
#pragma unroll
    for (int n = 0; n < NV; ++n) {
        const bool live = t0 + n < cnt;
        const double sc = live ? ws.zscale[g + n] : 0.0;
#pragma unroll
        for (int e = 0; e < EPT; ++e) {
            const int i = tid + BT_THREADS * e;
            x[n][e] = (live && i < M) ? ws.f[4][(size_t)i * N + g + n] * sc : 0.0;
        }
    }
    const double* G = Gws + (size_t)s * M * M;
    const double* tau = ws.tau + (size_t)s * M;
    // reflectors k, k-1, .., k-D+1 in flight: at small M one reflector's arithmetic is shorter than an L2 round trip
    constexpr int D = EPT <= 2 ? 4 : (EPT <= 4 ? 3 : (EPT <= 16 ? 2 : 1));
    double vq[D][EPT];
    int k = M - 3;
#pragma unroll
    for (int q = 0; q < D; ++q) {
#pragma unroll
        for (int e = 0; e < EPT; ++e) {
            const int i = tid + BT_THREADS * e, kk = k - q;
            vq[q][e] = (kk >= 0 && i > kk && i < M) ? __ldg(G + (size_t)kk * M + i) : 0.0;
        }
    }
    for (; k >= 0; --k) {
        const double tk = __ldg(tau + k);
        double vc[EPT];
#pragma unroll
        for (int e = 0; e < EPT; ++e) vc[e] = vq[0][e];
#pragma unroll
        for (int q = 0; q + 1 < D; ++q) {
#pragma unroll
            for (int e = 0; e < EPT; ++e) vq[q][e] = vq[q + 1][e];
        }
#pragma unroll
        for (int e = 0; e < EPT; ++e) {  // reflector k - D
            const int i = tid + BT_THREADS * e, kk = k - D;
            vq[D - 1][e] = (kk >= 0 && i > kk && i < M) ? __ldg(G + (size_t)kk * M + i) : 0.0;
        }
        double acc[NV];
#pragma unroll
        for (int n = 0; n < NV; ++n) {
            double a = 0.0;
#pragma unroll
            for (int e = 0; e < EPT; ++e) a = fma(vc[e], x[n][e], a);
            acc[n] = a;
        }
        // NV warp sums at once: halving butterfly (NV - 1 shuffles) leaves lane l with the 32/NV-lane partial of value
        // n = l / (32 / NV), the remaining xor steps complete it; the shuffle / shared-memory queue, not FP64, bounds
        // this kernel, so the plain version (5 NV shuffles, 8 NV shared loads per thread) was 3 x slower
#pragma unroll
        for (int h = 16, cn = NV / 2; cn >= 1; h >>= 1, cn >>= 1) {
            const bool up = (lane & h) != 0;
#pragma unroll
            for (int r = 0; r < cn; ++r) {
                const double send = up ? acc[r] : acc[r + cn], keep = up ? acc[r + cn] : acc[r];
                acc[r] = keep + __shfl_xor_sync(0xffffffffu, send, h);
            }
        }
#pragma unroll
        for (int h = 16 / NV; h >= 1; h >>= 1) acc[0] += __shfl_xor_sync(0xffffffffu, acc[0], h);
        double(*pb)[NV] = part[k & 1];
        if ((lane & (32 / NV - 1)) == 0) pb[warp][lane / (32 / NV)] = acc[0];
        __syncthreads();
        // totals over the 8 warps: lane l adds the partials of value l % NV (fixed tree), then the NV totals are broadcast
        double t;
        if (NV == 8) {
            t = pb[lane >> 3][lane & 7] + pb[(lane >> 3) + 4][lane & 7];
            t += __shfl_xor_sync(0xffffffffu, t, 8);
            t += __shfl_xor_sync(0xffffffffu, t, 16);
        } else if (NV == 4) {
            t = pb[lane >> 2][lane & 3];
            t += __shfl_xor_sync(0xffffffffu, t, 4);
            t += __shfl_xor_sync(0xffffffffu, t, 8);
            t += __shfl_xor_sync(0xffffffffu, t, 16);
        } else {  // NV == 2: lanes 0..15 hold warp (lane >> 1), value (lane & 1)
            t = (lane < 16) ? pb[lane >> 1][lane & 1] : 0.0;
            t += __shfl_xor_sync(0xffffffffu, t, 2);
            t += __shfl_xor_sync(0xffffffffu, t, 4);
            t += __shfl_xor_sync(0xffffffffu, t, 8);
        }
        t *= tk;
#pragma unroll
        for (int n = 0; n < NV; ++n) {
            const double tsum = __shfl_sync(0xffffffffu, t, n);
#pragma unroll
            for (int e = 0; e < EPT; ++e) x[n][e] = fma(-tsum, vc[e], x[n][e]);
        }
    }
#pragma unroll
    for (int n = 0; n < NV; ++n) {
        if (t0 + n >= cnt) continue;
        double* out = V + (g + n) * (size_t)N + lo;
#pragma unroll
        for (int e = 0; e < EPT; ++e) {
            const int i = tid + BT_THREADS * e;
            if (i < M) out[i] = x[n][e];
        }
        if (tid == 0) eps[g + n] = ws.lam[g + n];
    }
}

}  // namespace pfsm
