// sytrd_blocked.cuh -- step 2 for wide windows (gamma = M/N = 0.2-0.3, "M <= 3000"):
// BLOCKED Householder tridiagonalization B_s = Q T Q^T of all slices at once (the LAPACK dsytrd / dlatrd recurrence, lower
// variant, restated for a batched persistent grid).
//
// A panel of NB columns is reduced WITHOUT touching the trailing matrix: column k = k0 + j of the panel needs
//     y = A0 v_j - V (W^T v_j) - W (V^T v_j),      w_j = tau y - (tau^2/2)(y . v_j) v_j
// where A0 is the trailing matrix as it stood when the panel started and V, W hold the panel's earlier v_t, w_t.  So the
// per-column pass over the trailing matrix only READS its lower triangle (4 (M-k)^2 bytes; the unblocked kernels read and
// write it: 8 (M-k)^2 for the lower-triangle one) -- the HBM-bound part is halved -- and the rank-2NB update
//     A <- A - V W^T - W V^T        (lower tiles of rows / columns >= k0 + NB)
// is ONE batched product per panel on the FP64 tensor pipe (gemm_tn_kernel<EPI_SUB>, X = [V | W], Y = [W | V], K = 2 NB).
//
// sytrd_panel_kernel: one cooperative launch per panel, C CTAs per slice, two per-SLICE barriers per column (slices are
// independent: while one slice synchronizes, the others keep streaming).  Per column:
//   phase 1 (every CTA of the slice, redundantly and bitwise identically, O(M) work from L2-resident vectors):
//     finish the previous column (w_{j-1} from y, its scalar c = (tau^2/2)(y.v)), form column k of the updated matrix
//     a = base' - tau v y[k] + 2 c v   (see phase 2), the Householder vector v_j of a[k+1:], tau_j, d_k, e_k;
//     then the symv pass over the CTA's share of A0's lower triangle (the tiles, in row-major order, are cut into C equal
//     runs; 32 x 32 tile per warp, tile column per lane, all 32 loads in flight), the CTA's rows of the panel dots V^T v,
//     W^T v; per-CTA sums to global; barrier 1
//   phase 2 (own 32-row blocks): y = sum over CTAs (their contributions to A0 v) - V (W^T v) - W (V^T v),
//     base'[i] = A0[i][k+1] - sum_{t<j} (V[i][t] W[k+1][t] + W[i][t] V[k+1][t]) - tau y[i]  (column k+1 of the updated matrix
//     up to the two terms that need the global scalar c), partial y.v; barrier 2.
// Tile partial sums are reduced in shared memory in a fixed order, then across the slice's C CTAs in a fixed order: no
// atomics on data, results are bitwise reproducible.  Reflector k goes to the (unused) upper part of row k (columns k+1 ..,
// leading 1 stored), tau / d / e to the TriWs vectors: the layout tri_backtransform_kernel and the other kernels of
// tridiag_eig.cuh expect.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "kernels.cuh"
#include "tridiag_eig.cuh"

namespace pfsm {

constexpr int SB_NB = 32;        // panel width (K of the trailing update = 2 SB_NB)
constexpr int SB_THREADS = 512;  // 16 warps
constexpr int SB_NW = SB_THREADS / 32;

struct SbWs {           // workspace of the blocked tridiagonalization (device pointers)
    double* VW;         // [P][M][2 NB]  row i = (v_0[i] .. v_{NB-1}[i], w_0[i] .. w_{NB-1}[i])
    double* WV;         // [P][M][2 NB]  row i = (w_0[i] .., v_0[i] ..): the other operand of the rank-2NB update
    double* ypart;      // [CTAs][M]     per-CTA contributions to A0 v (row and column parts of the CTA's tiles)
    double* y;          // [2][P][M]     y of the column, double-buffered by column parity
    double* base;       // [2][P][M]     base' of the column
    double* dots;       // [P][C][2 NB]  per-CTA partial V^T v, W^T v
    double* yv;         // [2][P][C]     per-CTA partial y . v
    unsigned int* sbar; // [P]           per-slice barrier counters (zeroed before every launch)
};

// barrier over the C CTAs of one slice: `cnt` counts arrivals monotonically, `phase` = barriers passed so far.
// bar.sync orders the CTA's writes before thread 0's release; the acquire + bar.sync order the other CTAs' writes before
// every thread's later reads (release / acquire at gpu scope are cumulative over the CTA barrier).
__device__ __forceinline__ void sb_slice_barrier(unsigned int* cnt, unsigned int& phase, int C) {
    __syncthreads();
    ++phase;
    if (threadIdx.x == 0) {
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(cnt) : "memory");
        const unsigned int target = phase * (unsigned int)C;
        unsigned int v;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(cnt) : "memory");
        } while (v < target);
    }
    __syncthreads();
}

// sum over the block in a fixed order (every CTA of a slice gets the same bits); red: SB_NW doubles
__device__ __forceinline__ double sb_block_sum(double v, double* red) {
    v = warp_sum(v);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
#pragma unroll
    for (int w = 0; w < SB_NW; ++w) s += red[w];
    return s;
}

// tile g of the active lower triangle in row-major order: row block R (relative), column block S <= R
__device__ __forceinline__ void sb_tile_rc(int g, int& R, int& S) {
    int r = (int)((sqrt(8.0 * (double)g + 1.0) - 1.0) * 0.5);
    while ((r + 1) * (r + 2) / 2 <= g) ++r;
    while (r * (r + 1) / 2 > g) --r;
    R = r;
    S = g - r * (r + 1) / 2;
}

// B_s (rows / columns lo .. lo+M-1 of A) -> G_s, full storage (the upper part is overwritten by reflectors later)
__global__ void sytrd_copy_kernel(const double* __restrict__ A, int64_t N, int32_t M, SliceTable tab,
                                  double* __restrict__ Gws, int32_t s_off) {
    const int s = s_off + blockIdx.y, i = blockIdx.x;
    const int lo = tab.lo[s];
    const double* a = A + (size_t)(lo + i) * N + lo;
    double* g = Gws + ((size_t)s * M + i) * M;
    for (int j = threadIdx.x; j < M; j += blockDim.x) g[j] = a[j];
}

// Dynamic shared memory: vA[Mp] vB[Mp] (v_j / v_{j-1}, ping-pong), abuf[Mp] (column k; reused as ycta, the CTA's
// contribution to A0 v, once v_j exists), slots[2 * 32 * slot_tiles], red[SB_NW * 64], coef[4 * SB_NB].  Mp = M rounded up to 32.
__host__ __device__ inline size_t sb_smem_bytes(int M, int slot_tiles) {
    const size_t Mp = (size_t)((M + 31) / 32) * 32;
    return (3 * Mp + (size_t)64 * slot_tiles + (size_t)SB_NW * 64 + 4 * SB_NB) * sizeof(double);
}

// tiles of a CTA at the first column: the slot count that lets every column run in one chunk
inline int sb_max_tiles_per_cta(int M, int C) {
    const int64_t nbk = (M + 31) / 32, T = nbk * (nbk + 1) / 2;
    return (int)((T + C - 1) / C) + 1;
}

__global__ void __launch_bounds__(SB_THREADS, 1)
sytrd_panel_kernel(double* __restrict__ Gws, int32_t M, TriWs ws, SbWs sb, int32_t P, int32_t s_off, int32_t C,
                   int32_t k0, int32_t ncols, int32_t slot_tiles) {
    extern __shared__ double sm[];
    const int Mp = (M + 31) / 32 * 32;
    double* vbuf0 = sm;
    double* vbuf1 = sm + Mp;
    double* abuf = sm + 2 * Mp;
    double* ycta = abuf;                               // (abuf is dead once v_j is formed)
    double* slots = sm + 3 * Mp;                       // per tile: 32 row sums then 32 column sums
    double* red = slots + (size_t)64 * slot_tiles;     // SB_NW x 64
    double* coef = red + SB_NW * 64;                   // (V^T v)[t], (W^T v)[t], V[k+1][t], W[k+1][t]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int sl = blockIdx.x / C, c = blockIdx.x - sl * C, s = s_off + sl;
    double* G = Gws + (size_t)s * M * M;
    const size_t so = (size_t)s * M;
    double* VW = sb.VW + so * (2 * SB_NB);
    double* WV = sb.WV + so * (2 * SB_NB);
    double* ypart = sb.ypart + (size_t)sl * C * M;   // per-CTA buffers are indexed by the launch's own CTA numbering
    double* dots = sb.dots + (size_t)sl * C * (2 * SB_NB);
    const int ncta = gridDim.x;
    unsigned int* bar = sb.sbar + s;
    unsigned int phase = 0;
    const int nbk = (M + 31) / 32;
    for (int i = tid; i < Mp; i += SB_THREADS) vbuf0[i] = vbuf1[i] = 0.0;
    __syncthreads();

    double tau_p = 0.0;  // tau of the previous column
    for (int j = 0; j <= ncols; ++j) {
        const int k = k0 + j;
        double* vn = (j & 1) ? vbuf1 : vbuf0;        // v_j
        const double* vp = (j & 1) ? vbuf0 : vbuf1;  // v_{j-1}
        // ---------------- phase 1a: finish column j-1, form column k of the updated matrix ----------------
        if (j > 0) {
            const double* yp = sb.y + ((size_t)((j - 1) & 1) * P + s) * M;
            const double* bp = sb.base + ((size_t)((j - 1) & 1) * P + s) * M;
            const double* yvp = sb.yv + (size_t)((j - 1) & 1) * ncta + (size_t)sl * C;
            double yi[8], bi[8];  // M <= 4096 = 8 x 512: every load of the thread is in flight before the first use
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const int i = k + tid + SB_THREADS * e;
                yi[e] = (i < M) ? __ldcg(yp + i) : 0.0;
                bi[e] = (i < M) ? __ldcg(bp + i) : 0.0;
            }
            const double yk = __ldcg(yp + k);
            double yv = 0.0;
            for (int q0 = 0; q0 < C; q0 += 8) {  // fixed order
                double x[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) x[u] = (q0 + u < C) ? __ldcg(yvp + q0 + u) : 0.0;
#pragma unroll
                for (int u = 0; u < 8; ++u) yv += x[u];
            }
            const double c_p = 0.5 * tau_p * tau_p * yv;  // c = (tau^2 / 2)(y . v) of the previous column
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const int i = k + tid + SB_THREADS * e;
                if (i < M) {
                    const double v = vp[i];
                    const double w = fma(tau_p, yi[e], -c_p * v);
                    abuf[i] = bi[e] - tau_p * v * yk + 2.0 * c_p * v;
                    if ((i >> 5) % C == c) {  // own rows: the panel operands of the trailing update and of the later columns
                        const size_t o = (size_t)i * (2 * SB_NB);
                        __stcg(VW + o + (j - 1), v);
                        __stcg(VW + o + SB_NB + (j - 1), w);
                        __stcg(WV + o + (j - 1), w);
                        __stcg(WV + o + SB_NB + (j - 1), v);
                    }
                }
            }
        } else {
#pragma unroll
            for (int e = 0; e < 8; ++e) {  // column k0 (all updates applied)
                const int i = k + tid + SB_THREADS * e;
                if (i < M) abuf[i] = __ldcg(G + (size_t)i * M + k);
            }
        }
        __syncthreads();
        if (j == ncols) {
            // the panel is complete (VW / WV hold every column); the last panel also delivers the last diagonal entry
            if (k == M - 1 && c == 0 && tid == 0) {
                ws.d[so + k] = abuf[k];
                ws.e[so + k] = 0.0;
            }
            break;
        }
        // ---------------- phase 1b: Householder vector of a[k+1:] ----------------
        double acc = 0.0;
        for (int i = k + 2 + tid; i < M; i += SB_THREADS) acc = fma(abuf[i], abuf[i], acc);
        const double xn2 = sb_block_sum(acc, red);
        const double dk = abuf[k], alpha = abuf[k + 1];
        double tau = 0.0, beta = alpha, scal = 0.0;
        if (xn2 > 0.0) {
            beta = -copysign(sqrt(fma(alpha, alpha, xn2)), alpha);
            tau = (beta - alpha) / beta;
            scal = 1.0 / (alpha - beta);
        }
        for (int i = tid; i < M; i += SB_THREADS) vn[i] = (i <= k) ? 0.0 : ((i == k + 1) ? 1.0 : abuf[i] * scal);
        __syncthreads();
        if (c == 0) {
            for (int i = k + 1 + tid; i < M; i += SB_THREADS) G[(size_t)k * M + i] = vn[i];  // reflector k
            if (tid == 0) {
                ws.d[so + k] = dk;
                ws.e[so + k] = beta;
                ws.tau[so + k] = tau;
            }
        }
        const int b0 = (k + 1) >> 5;
        const int rb_first = b0 + ((c - b0) % C + C) % C;  // own 32-row blocks: rb_first, rb_first + C, ...
        // ---------------- phase 1c: own rows of the panel dots V^T v, W^T v (t < j) ----------------
        if (j > 0) {
            double av = 0.0, aw = 0.0;  // lane t: sum_i V[i][t] v[i], sum_i W[i][t] v[i] over this warp's rows
            for (int rbg = rb_first; rbg < nbk; rbg += 8 * C) {  // groups of 8 own blocks: 16 rows per warp, all loads first
                double xv[16], xw[16];
#pragma unroll
                for (int u = 0; u < 16; ++u) {
                    const int i = 32 * (rbg + (u >> 1) * C) + warp + SB_NW * (u & 1);
                    const bool ok = i > k && i < M;
                    xv[u] = ok ? __ldcg(VW + (size_t)i * (2 * SB_NB) + lane) : 0.0;
                    xw[u] = ok ? __ldcg(VW + (size_t)i * (2 * SB_NB) + SB_NB + lane) : 0.0;
                }
#pragma unroll
                for (int u = 0; u < 16; ++u) {
                    const int i = 32 * (rbg + (u >> 1) * C) + warp + SB_NW * (u & 1);
                    const double vi = (i < M) ? vn[i] : 0.0;
                    av = fma(xv[u], vi, av);
                    aw = fma(xw[u], vi, aw);
                }
            }
            red[warp * 64 + lane] = av;
            red[warp * 64 + 32 + lane] = aw;
            __syncthreads();
            if (tid < 64) {
                double t = 0.0;
#pragma unroll
                for (int w = 0; w < SB_NW; ++w) t += red[w * 64 + tid];
                __stcg(dots + (size_t)c * (2 * SB_NB) + tid, ((tid & 31) < j) ? t : 0.0);
            }
        }
        // ---------------- phase 1d: symv over this CTA's share of A0's lower triangle ----------------
        // the T tiles of the active triangle (row-major order) are cut into C equal contiguous runs
        for (int i = tid; i < Mp; i += SB_THREADS) ycta[i] = 0.0;
        if (tid < 256 && k + 1 < M) {  // phase 2 reads A0[i][k+1] of the own rows (a strided column): HBM -> L2 under the pass
            const int i = 32 * (rb_first + (tid >> 5) * C) + (tid & 31);
            if (i > k && i < M) asm volatile("prefetch.global.L2 [%0];" ::"l"(G + (size_t)i * M + k + 1));
        }
        const int nbr = nbk - b0;
        const int T = nbr * (nbr + 1) / 2;
        const int g_lo = (int)((int64_t)c * T / C), g_hi = (int)((int64_t)(c + 1) * T / C);
        for (int sub0 = g_lo; sub0 < g_hi; sub0 += slot_tiles) {  // (one pass unless the run outgrows the slots)
            const int sub1 = min(g_hi, sub0 + slot_tiles);
            __syncthreads();  // slots of the previous pass are no longer read; ycta is zeroed
            for (int g = sub0 + warp; g < sub1; g += SB_NW) {
                int R, S;
                sb_tile_rc(g, R, S);
                const int jc = 32 * (b0 + S) + lane, ib = 32 * (b0 + R);
                const double vnj = vn[jc];  // (vn is zero up to k and beyond M: Mp entries)
                double* slot = slots + (size_t)64 * (g - sub0);
                double b[32];
                double colacc = 0.0;
                if (S < R && ib + 32 <= M) {  // interior tile: every entry is below the diagonal
                    const double* gp = G + (size_t)ib * M + jc;
#pragma unroll
                    for (int r = 0; r < 32; ++r) b[r] = __ldg(gp + (size_t)r * M);
                    if (g + SB_NW < sub1) {
                        // the warp's next tile: HBM -> L2 now, under this tile's loads and arithmetic (lane = row, 256 bytes)
                        int Rn, Sn;
                        sb_tile_rc(g + SB_NW, Rn, Sn);
                        const int in = 32 * (b0 + Rn) + lane;
                        if (in < M) {
                            const double* pn = G + (size_t)in * M + 32 * (b0 + Sn);
                            asm volatile("prefetch.global.L2 [%0];" ::"l"(pn));
                            asm volatile("prefetch.global.L2 [%0];" ::"l"(pn + 16));
                        }
                    }
#pragma unroll
                    for (int r = 0; r < 32; ++r) {
                        colacc = fma(b[r], vn[ib + r], colacc);
                        b[r] *= vnj;
                    }
                } else {
#pragma unroll
                    for (int r = 0; r < 32; ++r) {
                        const int i = ib + r;
                        b[r] = (i < M && jc <= i) ? __ldg(G + (size_t)i * M + jc) : 0.0;
                    }
#pragma unroll
                    for (int r = 0; r < 32; ++r) {
                        const int i = ib + r;
                        if (jc < i) colacc = fma(b[r], vn[i], colacc);  // (b = 0 beyond M)
                        b[r] *= vnj;
                    }
                }
                // row sums: transposed butterfly, 31 shuffles; lane l ends with the sum of row ib + l
#pragma unroll
                for (int h = 16; h >= 1; h >>= 1) {
                    const bool up = (lane & h) != 0;
#pragma unroll
                    for (int r = 0; r < h; ++r) {
                        const double send = up ? b[r] : b[r + h], keep = up ? b[r + h] : b[r];
                        b[r] = keep + __shfl_xor_sync(0xffffffffu, send, h);
                    }
                }
                slot[lane] = b[0];
                slot[32 + lane] = colacc;
            }
            __syncthreads();
            // fold the pass into ycta in a fixed order: entry i takes the row sums of its row block's tiles, then the
            // column sums of its column block's tiles, each in ascending tile order
            int R0, S0, R1, S1;
            sb_tile_rc(sub0, R0, S0);
            sb_tile_rc(sub1 - 1, R1, S1);
            for (int i = 32 * b0 + tid; i < M; i += SB_THREADS) {
                const int R = (i >> 5) - b0, li = i & 31;
                double t = ycta[i];
                if (R >= R0 && R <= R1) {
                    const int ga = max(R * (R + 1) / 2, sub0), gb = min(R * (R + 1) / 2 + R + 1, sub1);
                    for (int g = ga; g < gb; ++g) t += slots[(size_t)64 * (g - sub0) + li];
                }
                for (int R2 = max(R, R0); R2 <= R1; ++R2) {
                    const int g = R2 * (R2 + 1) / 2 + R;
                    if (g >= sub0 && g < sub1) t += slots[(size_t)64 * (g - sub0) + 32 + li];
                }
                ycta[i] = t;
            }
        }
        __syncthreads();
        for (int i = k + 1 + tid; i < M; i += SB_THREADS) __stcg(ypart + (size_t)c * M + i, ycta[i]);
        sb_slice_barrier(bar, phase, C);
        // ---------------- phase 2: own 32-row blocks ----------------
        {
            double* yo = sb.y + ((size_t)(j & 1) * P + s) * M;
            double* bo = sb.base + ((size_t)(j & 1) * P + s) * M;
            // a pair of threads per row: the even one takes the V half of the row's panel entries, the odd one the W half.
            // Every load of a row is issued before its first use, and the loads of the first group of rows go out together
            // with those of the coefficients (panel dots, row k+1 of V and W): one L2 round trip serves both.
            double yvacc = 0.0;
            const int half = tid & 1, rs = tid >> 1;
            for (int rbg = rb_first; rbg < nbk || rbg == rb_first; rbg += 8 * C) {
                const int i = 32 * (rbg + (rs >> 5) * C) + (rs & 31);
                const bool ok = i > k && i < M;
                const double* row = VW + (size_t)(ok ? i : 0) * (2 * SB_NB) + half * SB_NB;
                double2 x[SB_NB / 2];
#pragma unroll
                for (int u = 0; u < SB_NB / 2; ++u)
                    x[u] = (ok && 2 * u < j) ? __ldcg(reinterpret_cast<const double2*>(row) + u) : make_double2(0.0, 0.0);
                double extra = 0.0;  // even: sum over the CTAs of the A0 v contributions; odd: A0[i][k+1]
                if (ok) {
                    if (half == 0) {
                        for (int q0 = 0; q0 < C; q0 += 8) {
                            double z[8];
#pragma unroll
                            for (int u = 0; u < 8; ++u) z[u] = (q0 + u < C) ? __ldcg(ypart + (size_t)(q0 + u) * M + i) : 0.0;
#pragma unroll
                            for (int u = 0; u < 8; ++u) extra += z[u];
                        }
                    } else {
                        extra = (k + 1 < M) ? __ldg(G + (size_t)i * M + k + 1) : 0.0;
                    }
                }
                if (rbg == rb_first) {
                    if (tid < 2 * SB_NB) {  // coefficients: the panel dots (sums over the CTAs, fixed order), row k+1 of V and W
                        const int t = tid & 31;
                        double a = 0.0;
                        if (j > 0 && t < j) {
                            for (int q0 = 0; q0 < C; q0 += 8) {
                                double xx[8];
#pragma unroll
                                for (int u = 0; u < 8; ++u) xx[u] = (q0 + u < C) ? __ldcg(dots + (size_t)(q0 + u) * (2 * SB_NB) + tid) : 0.0;
#pragma unroll
                                for (int u = 0; u < 8; ++u) a += xx[u];
                            }
                        }
                        coef[tid] = a;  // [0, 32): V^T v;  [32, 64): W^T v
                        coef[2 * SB_NB + tid] = (j > 0 && t < j) ? __ldcg(VW + (size_t)(k + 1) * (2 * SB_NB) + tid) : 0.0;  // V[k+1][t], W[k+1][t]
                    }
                    __syncthreads();
                }
                // even: s1 += V[i][t] (W^T v)[t], s2 += V[i][t] W[k+1][t];  odd: s1 += W[i][t] (V^T v)[t], s2 += W[i][t] V[k+1][t]
                const double* c1 = coef + (half ? 0 : SB_NB);
                const double* c2 = coef + 2 * SB_NB + (half ? 0 : SB_NB);
                double s1 = 0.0, s2 = 0.0;
#pragma unroll
                for (int u = 0; u < SB_NB / 2; ++u) {
                    s1 = fma(x[u].x, c1[2 * u], s1);
                    s1 = fma(x[u].y, c1[2 * u + 1], s1);
                    s2 = fma(x[u].x, c2[2 * u], s2);
                    s2 = fma(x[u].y, c2[2 * u + 1], s2);
                }
                s1 += __shfl_xor_sync(0xffffffffu, s1, 1);
                s2 += __shfl_xor_sync(0xffffffffu, s2, 1);
                const double other = __shfl_xor_sync(0xffffffffu, extra, 1);
                const double ysum = half ? other : extra, a0 = half ? extra : other;
                const double yi = ysum - s1;
                if (ok) {
                    if (half == 0) {
                        __stcg(yo + i, yi);
                        yvacc = fma(yi, vn[i], yvacc);
                    } else {
                        __stcg(bo + i, a0 - s2 - tau * yi);
                    }
                }
            }
            const double yvt = sb_block_sum(yvacc, red);
            if (tid == 0) __stcg(sb.yv + (size_t)(j & 1) * ncta + blockIdx.x, yvt);
        }
        tau_p = tau;
        sb_slice_barrier(bar, phase, C);
    }
}

}  // namespace pfsm
