// jacobi_smem.cuh -- step 2, shared-memory resident: one thread-block CLUSTER per slice.
//
// Same mathematics as jacobi_batched_kernel (one-sided Jacobi on G = B_s + sigma I, eigenvectors = normalized
// columns, mu = ||g|| - sigma), but the columns of G never leave shared memory.  The Mp = 2 h columns (M padded
// with zero "phantom" columns to a multiple of 2 CS) sit on the seats of a round-robin tournament,
//      top[0] top[1] ... top[h-1]
//      bot[0] bot[1] ... bot[h-1]          round r pairs (top[t], bot[t]) for every t
// and after every round all columns except top[0] move one seat along the cycle
//      top[1] -> top[2] -> ... -> top[h-1] -> bot[h-1] -> bot[h-2] -> ... -> bot[0] -> top[1].
// CTA k of the cluster owns seats t in [k h_loc, (k+1) h_loc).  Its top and bottom seats are ring buffers of
// h_loc + 1 column slots each, so "moving one seat" is a head-pointer increment; only the two columns that
// cross a CTA boundary are copied: the warp that rotated them stores the result straight into the spare slot
// of the neighbour's ring through distributed shared memory (mapa + st.shared::cluster), and the round ends
// with one cluster barrier (release/acquire).  Per round a CTA streams its 2 h_loc columns through the SM's
// own 128 B/clk shared-memory port instead of the chip-wide L2.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "kernels.cuh"

namespace pfsm {

__device__ __forceinline__ uint32_t mapa_shared(uint32_t addr, uint32_t cta) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(cta));
    return r;
}
__device__ __forceinline__ void st_cluster_f64(uint32_t addr, double v) {
    asm volatile("st.shared::cluster.f64 [%0], %1;" ::"r"(addr), "d"(v) : "memory");
}
__device__ __forceinline__ void st_cluster_s32(uint32_t addr, int v) {
    asm volatile("st.shared::cluster.s32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

// bytes of dynamic shared memory for (M, h_loc): column slots + ids + norms/ranks scratch
inline size_t jacobi_smem_bytes(int M, int h_loc) {
    const size_t nslots = 2 * (size_t)h_loc + 3;
    return nslots * M * sizeof(double) + nslots * sizeof(int) + 16 + (size_t)M * (sizeof(double) + sizeof(int)) + 64;
}

template <int EPL>
__global__ void __launch_bounds__(JACOBI_THREADS, 1)
jacobi_smem_kernel(const double* __restrict__ A, int64_t N, int32_t M, int32_t m, int32_t h_loc, SliceTable tab,
                   double* __restrict__ nrm_g, double* __restrict__ V, double* __restrict__ eps,
                   int* __restrict__ rotcnt, unsigned long long* info) {
    const int CS = (int)cluster_nctarank(), cr = (int)cluster_ctarank();
    const int s = blockIdx.x / CS;
    const int lo = tab.lo[s], off = tab.off[s], g0 = tab.g0[s];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    constexpr int NW = JACOBI_THREADS / 32;
    const int h = h_loc * CS, Mp = 2 * h;
    int* rot = rotcnt + (size_t)s * JACOBI_MAX_SWEEPS;
    double* nrm_s = nrm_g + (size_t)s * Mp;  // global scratch: final column norms by column id

    extern __shared__ __align__(16) unsigned char smem_jac[];
    const int nslots = 2 * h_loc + 3;
    double* cols = reinterpret_cast<double*>(smem_jac);                 // cols[slot][M]
    int* ids = reinterpret_cast<int*>(cols + (size_t)nslots * M);       // column id held by each slot
    double* nrm = reinterpret_cast<double*>(ids + ((nslots + 3) & ~3)); // nrm[M], then rank[M]
    int* rank = reinterpret_cast<int*>(nrm + M);
    __shared__ double red[NW];
    __shared__ double s_sigma;

    // slot map.  slot 0: the fixed column (used by CTA 0 only).  Top ring: slots T0 .. T0+h_loc (CTA 0 uses a
    // ring of h_loc slots for its h_loc-1 moving top seats).  Bottom ring: slots B0 .. B0+h_loc.
    const int T0 = 1, B0 = 2 + h_loc;
    const int RT = h_loc + 1;                   // ring size of a standard top ring and of every bottom ring
    const int RT0 = h_loc;                      // ring size of CTA 0's top ring
    int head_t = 0, head_t0 = 0, head_b = 0;    // identical on every CTA of every cluster (pure functions of the round)
    // heads stay in [0, ring size) and seats in [0, h_loc], so one conditional subtraction replaces the modulo
    auto wrap = [](int v, int ring) -> int { return v >= ring ? v - ring : v; };
    auto slot_top = [&](int t) -> int {
        if (cr == 0) return t == 0 ? 0 : T0 + wrap(head_t0 + t - 1, RT0);
        return T0 + wrap(head_t + t, RT);
    };
    auto slot_bot = [&](int t) -> int { return B0 + wrap(head_b + t, RT); };

    // ---- Gershgorin shift (every CTA computes the same sigma) ----
    double bound = 0.0;
    for (int r = tid; r < M; r += JACOBI_THREADS) {
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

    // ---- initial seating: top[t] = column t, bot[t] = column h + t (global seat t = cr h_loc + tl) ----
    for (int q = warp; q < 2 * h_loc; q += NW) {
        const bool is_top = q < h_loc;
        const int tl = is_top ? q : q - h_loc;
        const int cid = (is_top ? 0 : h) + cr * h_loc + tl;
        const int slot = is_top ? slot_top(tl) : slot_bot(tl);
        double* dst = cols + (size_t)slot * M;
        for (int r = lane; r < M; r += 32) {
            double v = 0.0;
            if (cid < M) {
                v = A[(size_t)(lo + cid) * N + lo + r];
                if (r == cid) v += sigma;
            }
            dst[r] = v;
        }
        if (lane == 0) ids[slot] = cid;
    }
    if (CS > 1) cluster_sync_all(); else __syncthreads();

    const uint32_t cols_u32 = (uint32_t)__cvta_generic_to_shared(cols);
    const uint32_t ids_u32 = (uint32_t)__cvta_generic_to_shared(ids);
    const int nrounds = Mp - 1;
    const double tol2 = 2.220446049250313e-16 * 2.220446049250313e-16 * (double)M;  // (sqrt(M) eps)^2
    bool converged = false;
    for (int sweep = 0; sweep < JACOBI_MAX_SWEEPS; ++sweep) {
        int nrot = 0;
        for (int rnd = 0; rnd < nrounds; ++rnd) {
            for (int t = warp; t < h_loc; t += NW) {
                const int sp = slot_top(t), sq = slot_bot(t);
                double* gp = cols + (size_t)sp * M;
                double* gq = cols + (size_t)sq * M;
                double x[EPL], y[EPL];
                double aa = 0.0, bb = 0.0, ab = 0.0;
#pragma unroll
                for (int e = 0; e < EPL; ++e) {
                    const int r = lane + 32 * e;
                    x[e] = (r < M) ? gp[r] : 0.0;
                    y[e] = (r < M) ? gq[r] : 0.0;
                    aa = fma(x[e], x[e], aa);
                    bb = fma(y[e], y[e], bb);
                    ab = fma(x[e], y[e], ab);
                }
                aa = warp_sum(aa);
                bb = warp_sum(bb);
                ab = warp_sum(ab);
                const bool rotate = ab * ab > tol2 * (aa * bb);  // |g_p . g_q| > sqrt(M) eps ||g_p|| ||g_q||
                if (rotate) {
                    const double zeta = (bb - aa) / (2.0 * ab);
                    const double tt = copysign(1.0, zeta) / (fabs(zeta) + sqrt(fma(zeta, zeta, 1.0)));
                    const double cs = rsqrt(fma(tt, tt, 1.0)), sn = cs * tt;
#pragma unroll
                    for (int e = 0; e < EPL; ++e) {
                        const double xe = x[e], ye = y[e];
                        x[e] = cs * xe - sn * ye;
                        y[e] = sn * xe + cs * ye;
                    }
                    ++nrot;
                }
                // where do the two columns sit next round?  top[t] -> top[t+1] (same slot) unless it is the
                // CTA's last top seat; bot[t] -> bot[t-1] (same slot) unless it is the CTA's first bottom seat.
                const bool top_fixed = (cr == 0 && t == 0);
                const bool top_leaves = (t == h_loc - 1) && !top_fixed;
                const bool bot_leaves = (t == 0);
                // destination of a leaving top column: right neighbour's top spare, or (last CTA) own bottom spare
                uint32_t dst_cta = (uint32_t)cr;
                int dst_slot = sp;
                if (top_leaves) {
                    if (cr < CS - 1) {
                        dst_cta = (uint32_t)(cr + 1);
                        dst_slot = T0 + wrap(head_t + RT - 1, RT);
                    } else {
                        dst_slot = B0 + wrap(head_b + h_loc, RT);
                    }
                }
                if (top_leaves) {
                    const uint32_t base = mapa_shared(cols_u32 + (uint32_t)((size_t)dst_slot * M * 8), dst_cta);
#pragma unroll
                    for (int e = 0; e < EPL; ++e) {
                        const int r = lane + 32 * e;
                        if (r < M) st_cluster_f64(base + 8u * r, x[e]);
                    }
                    if (lane == 0) st_cluster_s32(mapa_shared(ids_u32 + 4u * dst_slot, dst_cta), ids[sp]);
                } else if (rotate) {
#pragma unroll
                    for (int e = 0; e < EPL; ++e) {
                        const int r = lane + 32 * e;
                        if (r < M) gp[r] = x[e];
                    }
                }
                // destination of a leaving bottom column: left neighbour's bottom spare, or (CTA 0) own top spare
                if (bot_leaves) {
                    uint32_t bcta = (uint32_t)cr;
                    int bslot;
                    if (cr > 0) {
                        bcta = (uint32_t)(cr - 1);
                        bslot = B0 + wrap(head_b + h_loc, RT);
                    } else {
                        bslot = T0 + wrap(head_t0 + RT0 - 1, RT0);
                    }
                    const uint32_t base = mapa_shared(cols_u32 + (uint32_t)((size_t)bslot * M * 8), bcta);
#pragma unroll
                    for (int e = 0; e < EPL; ++e) {
                        const int r = lane + 32 * e;
                        if (r < M) st_cluster_f64(base + 8u * r, y[e]);
                    }
                    if (lane == 0) st_cluster_s32(mapa_shared(ids_u32 + 4u * bslot, bcta), ids[sq]);
                } else if (rotate) {
#pragma unroll
                    for (int e = 0; e < EPL; ++e) {
                        const int r = lane + 32 * e;
                        if (r < M) gq[r] = y[e];
                    }
                }
            }
            if (rnd == nrounds - 1 && lane == 0 && nrot) atomicAdd(rot + sweep, nrot);
            if (CS > 1) cluster_sync_all(); else __syncthreads();
            head_t = wrap(head_t + RT - 1, RT);
            head_t0 = wrap(head_t0 + RT0 - 1, RT0);
            head_b = wrap(head_b + 1, RT);
        }
        const int total = __ldcg(rot + sweep);
        if (total == 0) {
            converged = true;
            break;
        }
    }
    if (!converged && tid == 0 && cr == 0) atomicMin(info, (unsigned long long)(N + s + 1));

    // ---- norms of this CTA's columns -> global scratch by column id; then every CTA ranks and writes its own ----
    for (int q = warp; q < 2 * h_loc; q += NW) {
        const int slot = q < h_loc ? slot_top(q) : slot_bot(q - h_loc);
        const int cid = ids[slot];
        const double* gc = cols + (size_t)slot * M;
        double ss = 0.0;
        for (int r = lane; r < M; r += 32) ss = fma(gc[r], gc[r], ss);
        ss = warp_sum(ss);
        if (lane == 0 && cid < M) nrm_s[cid] = sqrt(ss);
    }
    __threadfence();
    if (CS > 1) cluster_sync_all(); else __syncthreads();
    for (int c = tid; c < M; c += JACOBI_THREADS) nrm[c] = __ldcg(nrm_s + c);
    __syncthreads();
    for (int c = tid; c < M; c += JACOBI_THREADS) {
        const double v = nrm[c];
        int rk = 0;
        for (int j = 0; j < M; ++j) {
            const double u = nrm[j];
            rk += (u < v || (u == v && j < c)) ? 1 : 0;
        }
        rank[c] = rk;
    }
    __syncthreads();
    for (int q = warp; q < 2 * h_loc; q += NW) {
        const int slot = q < h_loc ? slot_top(q) : slot_bot(q - h_loc);
        const int cid = ids[slot];
        if (cid >= M) continue;
        const int j = rank[cid] - off;
        if (j < 0 || j >= m) continue;
        const double nv = nrm[cid];
        const double inv = 1.0 / nv;
        const double* gc = cols + (size_t)slot * M;
        double* v = V + (size_t)(g0 + j) * N + lo;
        for (int r = lane; r < M; r += 32) v[r] = gc[r] * inv;
        if (lane == 0) eps[g0 + j] = nv - sigma;
    }
}

}  // namespace pfsm
