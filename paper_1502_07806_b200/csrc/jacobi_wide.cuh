// jacobi_wide.cuh -- step 2 for wide windows: submatrix order 512 < M <= 4096, the regime the paper
// recommends (gamma = M/N = 0.2-0.3, "M <= 3000").
//
// Same mathematics as the other two step-2 kernels (one-sided Jacobi on G = B_s + sigma I, eigenvectors = normalized
// columns, mu = ||g|| - sigma, ranks by counting), but a column no longer fits the registers of one warp and the batch
// of P submatrices (8 P M^2 bytes: 0.1-1 GB) no longer fits shared memory or L2:
//   * ONE persistent cooperative grid works on all slices at once.  The unit of work is (slice, column pair of the
//     current tournament round); units are dealt round-robin to "pair groups" of 256 threads (two per CTA), so the
//     load is even whatever P is, and rounds are separated by a grid-wide barrier (monotonic counter, one atomic per
//     CTA, ld.acquire spin) instead of a per-slice cluster barrier.
//   * A group keeps both columns of its pair in registers (EPT doubles per thread per column, M <= 256 EPT), reduces
//     the three dot products with shuffles + one 256-thread named barrier (double-buffered partials), rotates, and
//     writes back.  G lives in the handle's workspace: every round streams it once (read + write, 16 P M^2 bytes):
//     the kernel is bound by L2 / HBM bandwidth, and a sweep costs (M - 1) such rounds.
//   * A slice whose sweep made no rotation is finished; its units are skipped from then on.  The kernel ends when every
//     slice of the launch has finished (or at the sweep cap: info = N + s + 1 as in the other kernels).
// Every pair of a round is disjoint and every reduction has a fixed order: results are bitwise reproducible.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "kernels.cuh"

namespace pfsm {

constexpr int JW_THREADS = 512;  // per CTA
constexpr int JW_GROUP = 256;    // threads that share one column pair
constexpr int JW_GPC = JW_THREADS / JW_GROUP;
constexpr int JW_MAX_M = 4096;   // 256 threads x 16 doubles per column

// grid-wide barrier: `bar` counts arrivals monotonically (zeroed before the launch); `phase` = barriers passed so far
__device__ __forceinline__ void jw_grid_barrier(unsigned int* bar, unsigned int& phase) {
    __syncthreads();
    ++phase;
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(bar, 1u);
        const unsigned int target = phase * gridDim.x;
        unsigned int v;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
        } while (v < target);
        __threadfence();
    }
    __syncthreads();
}

__device__ __forceinline__ void jw_group_sync(int g) {  // named barrier 1 + g over the group's 256 threads
    asm volatile("bar.sync %0, %1;" ::"r"(1 + g), "n"(JW_GROUP) : "memory");
}

// ws: per slice (M + 16) doubles: column norms [0, M), sigma at [M]  (the handle's nrm_g)
template <int EPT>
__global__ void __launch_bounds__(JW_THREADS, 1)
jacobi_wide_kernel(const double* __restrict__ A, int64_t N, int32_t M, SliceTable tab, double* __restrict__ Gws,
                   double* __restrict__ ws, double* __restrict__ V, double* __restrict__ eps,
                   int* __restrict__ rotcnt, unsigned long long* info, int32_t s_off, int32_t ns,
                   unsigned int* __restrict__ bar) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int grp = tid / JW_GROUP, gt = tid % JW_GROUP, gwarp = gt >> 5;
    const int gidx = blockIdx.x * JW_GPC + grp, ngroups = gridDim.x * JW_GPC;
    const int gw = blockIdx.x * (JW_THREADS / 32) + warp, nwarps = gridDim.x * (JW_THREADS / 32);
    const size_t wss = (size_t)M + 16;
    unsigned int phase = 0;

    __shared__ double red[JW_THREADS / 32];
    __shared__ double part[2][JW_GPC][JW_GROUP / 32][3];
    extern __shared__ int done[];  // ns flags: slice finished

    // Gershgorin bound of every slice (CTA per slice; thread per row, consecutive rows contiguous) -> sigma
    for (int sl = blockIdx.x; sl < ns; sl += gridDim.x) {
        const int lo = tab.lo[s_off + sl];
        double bound = 0.0;
        for (int r = tid; r < M; r += JW_THREADS) {
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
            for (int w = 0; w < JW_THREADS / 32; ++w) b = fmax(b, red[w]);
            ws[(size_t)(s_off + sl) * wss + M] = (b > 0.0) ? 2.0 * b : 1.0;
        }
        __syncthreads();
    }
    for (int i = tid; i < ns; i += JW_THREADS) done[i] = 0;
    jw_grid_barrier(bar, phase);

    // G = B_s + sigma I (column c of G = row lo + c of A, contiguous)
    for (int u = gw; u < ns * M; u += nwarps) {
        const int sl = u / M, c = u - sl * M, s = s_off + sl;
        const int lo = tab.lo[s];
        const double sigma = __ldcg(ws + (size_t)s * wss + M);
        const double* a = A + (size_t)(lo + c) * N + lo;
        double* g = Gws + ((size_t)s * M + c) * M;
        for (int r = lane; r < M; r += 32) g[r] = a[r] + (r == c ? sigma : 0.0);
    }
    jw_grid_barrier(bar, phase);

    const int Me = M + (M & 1);  // phantom column when M is odd
    const int n1 = Me - 1, npairs = Me / 2;
    const double tol = 2.220446049250313e-16 * sqrt((double)M);
    int it = 0;  // pairs this group has reduced (selects the partials buffer)
    int sweep = 0, left = ns;
    for (; sweep < JACOBI_MAX_SWEEPS && left > 0; ++sweep) {
        for (int rnd = 0; rnd < n1; ++rnd) {
            for (int u = gidx; u < ns * npairs; u += ngroups) {
                const int sl = u / npairs, pi = u - sl * npairs;
                if (done[sl]) continue;
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
                const int s = s_off + sl;
                double* gp = Gws + ((size_t)s * M + p) * M;
                double* gq = Gws + ((size_t)s * M + q) * M;
                double x[EPT], y[EPT];
#pragma unroll
                for (int e = 0; e < EPT; ++e) {
                    const int r = gt + JW_GROUP * e;
                    x[e] = (r < M) ? __ldcg(gp + r) : 0.0;
                    y[e] = (r < M) ? __ldcg(gq + r) : 0.0;
                }
                double aa = 0.0, bb = 0.0, ab = 0.0;
#pragma unroll
                for (int e = 0; e < EPT; ++e) {
                    aa = fma(x[e], x[e], aa);
                    bb = fma(y[e], y[e], bb);
                    ab = fma(x[e], y[e], ab);
                }
                aa = warp_sum(aa);
                bb = warp_sum(bb);
                ab = warp_sum(ab);
                double(*pb)[3] = part[it & 1][grp];
                ++it;
                if (lane == 0) {
                    pb[gwarp][0] = aa;
                    pb[gwarp][1] = bb;
                    pb[gwarp][2] = ab;
                }
                jw_group_sync(grp);
                aa = bb = ab = 0.0;
#pragma unroll
                for (int w = 0; w < JW_GROUP / 32; ++w) {
                    aa += pb[w][0];
                    bb += pb[w][1];
                    ab += pb[w][2];
                }
                if (fabs(ab) > tol * sqrt(aa * bb)) {
                    const double zeta = (bb - aa) / (2.0 * ab);
                    const double tt = copysign(1.0, zeta) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
                    const double cs = 1.0 / sqrt(1.0 + tt * tt), sn = cs * tt;
#pragma unroll
                    for (int e = 0; e < EPT; ++e) {
                        const int r = gt + JW_GROUP * e;
                        if (r < M) {
                            gp[r] = cs * x[e] - sn * y[e];
                            gq[r] = sn * x[e] + cs * y[e];
                        }
                    }
                    if (gt == 0) atomicAdd(rotcnt + (size_t)s * JACOBI_MAX_SWEEPS + sweep, 1);
                }
            }
            jw_grid_barrier(bar, phase);
        }
        // a slice whose sweep rotated nothing is finished (every CTA reads the same counters -> same flags)
        __syncthreads();
        for (int i = tid; i < ns; i += JW_THREADS)
            if (!done[i] && __ldcg(rotcnt + (size_t)(s_off + i) * JACOBI_MAX_SWEEPS + sweep) == 0) done[i] = 1;
        __syncthreads();
        left = 0;
        for (int i = 0; i < ns; ++i) left += done[i] ? 0 : 1;
    }
    if (left > 0 && blockIdx.x == 0)
        for (int i = tid; i < ns; i += JW_THREADS)
            if (!done[i]) atomicMin(info, (unsigned long long)(N + s_off + i + 1));

    // column norms -> ws
    for (int u = gw; u < ns * M; u += nwarps) {
        const int sl = u / M, c = u - sl * M, s = s_off + sl;
        const double* gc = Gws + ((size_t)s * M + c) * M;
        double ss = 0.0;
        for (int r = lane; r < M; r += 32) {
            const double g = __ldcg(gc + r);
            ss = fma(g, g, ss);
        }
        ss = warp_sum(ss);
        if (lane == 0) ws[(size_t)s * wss + c] = sqrt(ss);
    }
    jw_grid_barrier(bar, phase);

    // rank by counting (ties: lower column index first); the slice's m eigenpairs go to V and eps
    for (int u = gw; u < ns * M; u += nwarps) {
        const int sl = u / M, c = u - sl * M, s = s_off + sl;
        const double* nrm = ws + (size_t)s * wss;
        const double nv = __ldcg(nrm + c);
        int rk = 0;
        for (int j = lane; j < M; j += 32) {
            const double w = __ldcg(nrm + j);
            rk += (w < nv || (w == nv && j < c)) ? 1 : 0;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) rk += __shfl_xor_sync(0xffffffffu, rk, o);
        const int j = rk - tab.off[s];
        if (j < 0 || j >= tab.cnt[s]) continue;
        const int lo = tab.lo[s], g0 = tab.g0[s];
        const double inv = 1.0 / nv;
        const double* gc = Gws + ((size_t)s * M + c) * M;
        double* v = V + (size_t)(g0 + j) * N + lo;
        for (int r = lane; r < M; r += 32) v[r] = __ldcg(gc + r) * inv;
        if (lane == 0) eps[g0 + j] = nv - __ldcg(nrm + M);
    }
}

}  // namespace pfsm
