// jacobi_smem.cuh -- step 2, shared-memory resident: one thread-block CLUSTER per slice.  Product path for
// submatrix orders M < 16; second route (option step2_route = 1) up to M ~ 480.
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
// cross a CTA boundary are copied: the warp that rotated one sends it, straight from its registers, into the spare
// slot of the neighbour's ring through distributed shared memory with st.async, which completes its bytes on the
// receiver's mbarrier -- a point-to-point exchange that overlaps the CTA's other pairs; a cluster barrier is needed
// only once per sweep (convergence count).  Per round a CTA streams its 2 h_loc columns through the SM's own 128 B/clk
// shared-memory port instead of the chip-wide L2.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "gemm_tn.cuh"  // lds128
#include "kernels.cuh"

namespace pfsm {

__device__ __forceinline__ uint32_t mapa_shared(uint32_t addr, uint32_t cta) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(cta));
    return r;
}
// remote shared-memory store whose completion is counted (in bytes) on the destination CTA's mbarrier
__device__ __forceinline__ void st_async_v2f64(uint32_t raddr, double2 v, uint32_t rmbar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f64 [%0], {%1,%2}, [%3];" ::"r"(raddr),
                 "d"(v.x), "d"(v.y), "r"(rmbar)
                 : "memory");
}
__device__ __forceinline__ void st_async_f64(uint32_t raddr, double v, uint32_t rmbar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.f64 [%0], %1, [%2];" ::"r"(raddr), "d"(v),
                 "r"(rmbar)
                 : "memory");
}
__device__ __forceinline__ void st_async_s32(uint32_t raddr, int v, uint32_t rmbar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.s32 [%0], %1, [%2];" ::"r"(raddr), "r"(v),
                 "r"(rmbar)
                 : "memory");
}
__device__ __forceinline__ void sts128(uint32_t addr, double2 v) {
    asm volatile("st.shared.v2.f64 [%0], {%1,%2};" ::"r"(addr), "d"(v.x), "d"(v.y) : "memory");
}

// Inline FP64 reciprocal square root for well-scaled positive arguments (column norms and their
// combinations: no zeros, infinities or subnormals): FP32 seed + two Newton steps (24 -> 48 -> 96 bits), about 8
// instructions each instead of the library's call with its special-case handling.
__device__ __forceinline__ double fast_rsqrt_pos(double x) {
    double y = (double)rsqrtf((float)x);
    const double hx = 0.5 * x;
    y = y * fma(-hx * y, y, 1.5);
    y = y * fma(-hx * y, y, 1.5);
    return y;
}

// bytes of dynamic shared memory for (M, h_loc): column slots + ids + norms/ranks scratch
inline int jacobi_padded_rows(int M) { return (M + 63) / 64 * 64; }  // column slot length: whole double2 per lane
inline size_t jacobi_smem_bytes(int M, int h_loc) {
    const size_t nslots = 2 * (size_t)h_loc + 3;
    return nslots * jacobi_padded_rows(M) * sizeof(double) + nslots * sizeof(double) + nslots * sizeof(int) + 16 + (size_t)M * (sizeof(double) + sizeof(int)) + 64;
}

// Threads per CTA.  A warp keeps both columns of its pair in registers (2 EPL doubles per lane): with 1024 threads the
// register file allows 64 per thread, which holds EPL <= 8 (M <= 256); wider columns get 512 threads (128 registers)
// and a warp takes two pairs per round instead of spilling the columns to local memory (measured at 13 slices, per
// round: M = 416 6.6 -> 3.1 us, M = 384 3.7 -> 2.9 us; at EPL = 10 the 64-byte spill of the 1024-thread build is faster).
__host__ __device__ constexpr int jacobi_smem_threads(int epl) { return epl <= 10 ? 1024 : 512; }

// HALF (EPL <= 8 only): 512 threads and 64 registers, so two CTAs -- of two different slices -- share an SM and one
// fills the other's barrier and exchange waits.  Chosen when the slices need more than one wave anyway
// (choose_jacobi_layout; config 4: 64 clusters of 8 half CTAs 12.5 ms vs 64 clusters of 4 full CTAs 13.4 ms).
template <int EPL, bool HALF = false>
__global__ void __launch_bounds__(HALF ? 512 : jacobi_smem_threads(EPL), HALF ? 2 : 1)
jacobi_smem_kernel(const double* __restrict__ A, int64_t N, int32_t M, int32_t h_loc, SliceTable tab,
                   double* __restrict__ nrm_g, double* __restrict__ V, double* __restrict__ eps,
                   int* __restrict__ rotcnt, unsigned long long* info, int32_t s_off, int32_t compact) {
    const int CS = (int)cluster_nctarank(), cr = (int)cluster_ctarank();
    const int s = s_off + blockIdx.x / CS;  // s_off: first slice of this launch
    const int lo = tab.lo[s], off = tab.off[s], g0 = tab.g0[s], m = tab.cnt[s];
    // the slice's submatrix B_s: a principal block of A (leading dimension N), or -- compact != 0 -- block s of a
    // packed P x M x M copy of the diagonal blocks (pfsm_solve_host uploads those first)
    const double* Ab = compact ? A + (size_t)s * M * M : A + (size_t)lo * N + lo;
    const int64_t ldb = compact ? (int64_t)M : N;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    constexpr int NT = HALF ? 512 : jacobi_smem_threads(EPL), NW = NT / 32;
    const int h = h_loc * CS, Mp = 2 * h;
    constexpr int Ms = 32 * EPL, E2 = EPL / 2;  // padded column length (rows M..Ms-1 are zero and stay zero)
    int* rot = rotcnt + (size_t)s * JACOBI_MAX_SWEEPS;
    double* nrm_s = nrm_g + (size_t)s * Mp;  // global scratch: final column norms by column id

    extern __shared__ __align__(16) unsigned char smem_jac[];
    const int nslots = 2 * h_loc + 3;
    double* cols = reinterpret_cast<double*>(smem_jac);                 // cols[slot][Ms]
    double* nrm2 = cols + (size_t)nslots * Ms;                                       // squared norm of the column in each slot
    int* ids = reinterpret_cast<int*>(nrm2 + nslots);                    // column id held by each slot
    double* nrm = reinterpret_cast<double*>(ids + ((nslots + 3) & ~3)); // nrm[M], then rank[M]
    int* rank = reinterpret_cast<int*>(nrm + M);
    __shared__ double red[NW];
    __shared__ double s_sigma;
    // incoming-column barriers: [2 dir + par], dir 0 = top column from the left CTA, 1 = bottom column from the right;
    // rounds alternate between the two barriers of a direction (par = round & 1), so a fast neighbour's next column can
    // never be counted into the phase this CTA is still waiting for
    __shared__ __align__(8) unsigned long long mbar_in[4];

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
    for (int r = tid; r < M; r += NT) {
        double sum = 0.0;
        for (int c = 0; c < M; ++c) sum += fabs(Ab[(size_t)c * ldb + r]);
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
        double* dst = cols + (size_t)slot * Ms;
        for (int r = lane; r < Ms; r += 32) {
            double v = 0.0;
            if (cid < M && r < M) {
                v = Ab[(size_t)cid * ldb + r];
                if (r == cid) v += sigma;
            }
            dst[r] = v;
        }
        if (lane == 0) ids[slot] = cid;
    }
    if (tid == 0) {
        for (int b = 0; b < 4; ++b) mbar_init((uint32_t)__cvta_generic_to_shared(&mbar_in[b]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (CS > 1) cluster_sync_all(); else __syncthreads();

    const uint32_t mbar_u32 = (uint32_t)__cvta_generic_to_shared(&mbar_in[0]);
    const bool has_left = cr > 0, has_right = cr < CS - 1;  // neighbours that exchange a column with this CTA every round
    const uint32_t col_tx = (uint32_t)(Ms * 8 + 8 + 4);   // bytes one incoming column (+ its squared norm and id) completes
    const uint32_t nrm2_u32 = (uint32_t)__cvta_generic_to_shared(nrm2);
    uint32_t rcount = 0;  // rounds done so far (all sweeps): barrier parity = rcount & 1, its phase bit = (rcount >> 1) & 1
    const uint32_t cols_u32 = (uint32_t)__cvta_generic_to_shared(cols);
    const uint32_t ids_u32 = (uint32_t)__cvta_generic_to_shared(ids);
    const int nrounds = Mp - 1;
    const double tol2 = 2.220446049250313e-16 * 2.220446049250313e-16 * (double)M;  // (sqrt(M) eps)^2
    bool converged = false;
    for (int sweep = 0; sweep < JACOBI_MAX_SWEEPS; ++sweep) {
        int nrot = 0;
        for (int rnd = 0; rnd < nrounds; ++rnd) {
            const uint32_t par = rcount & 1u;
            for (int t = warp; t < h_loc; t += NW) {
                const int sp = slot_top(t), sq = slot_bot(t);
                const uint32_t ap = cols_u32 + (uint32_t)(sp * Ms * 8) + 16u * lane;
                const uint32_t aq = cols_u32 + (uint32_t)(sq * Ms * 8) + 16u * lane;
                double2 x[E2], y[E2];
                double aa = 0.0, bb = 0.0, ab = 0.0;
                // Squared column norms travel with the columns and are updated analytically after a rotation
                // (||x'||^2 = aa - t ab, ||y'||^2 = bb + t ab); they are recomputed from the data in the first round of
                // every sweep, so rounding drift is bounded by one sweep.  They only steer the rotation angle and the
                // convergence test; the eigenvalues come from norms recomputed at the end.
                if (rnd == 0) {
#pragma unroll
                    for (int e = 0; e < E2; ++e) {  // lane holds rows 2 (lane + 32 e), +1: conflict-free 16-byte accesses
                        x[e] = lds128(ap + 512u * e);
                        y[e] = lds128(aq + 512u * e);
                        aa = fma(x[e].x, x[e].x, aa); aa = fma(x[e].y, x[e].y, aa);
                        bb = fma(y[e].x, y[e].x, bb); bb = fma(y[e].y, y[e].y, bb);
                        ab = fma(x[e].x, y[e].x, ab); ab = fma(x[e].y, y[e].y, ab);
                    }
                    aa = warp_sum(aa);
                    bb = warp_sum(bb);
                    ab = warp_sum(ab);
                } else {
                    double ab1 = 0.0;  // two independent accumulation chains halve the dependent-FMA latency
#pragma unroll
                    for (int e = 0; e < E2; ++e) {
                        x[e] = lds128(ap + 512u * e);
                        y[e] = lds128(aq + 512u * e);
                        ab = fma(x[e].x, y[e].x, ab);
                        ab1 = fma(x[e].y, y[e].y, ab1);
                    }
                    ab = warp_sum(ab + ab1);
                    aa = nrm2[sp];
                    bb = nrm2[sq];
                }
                // Boundary seats: read what travels with the column now, then meet the other boundary warp.  A column
                // sent to a neighbour lets that neighbour run ahead and overwrite, with ITS next column, the slot the
                // other boundary seat is reading from this round -- so neither boundary warp sends before both loaded.
                const bool boundary = (CS > 1) && (t == 0 || t == h_loc - 1);
                int idp = 0, idq = 0;
                if (t == 0 || t == h_loc - 1) {
                    idp = ids[sp];
                    idq = ids[sq];
                }
                if (boundary) asm volatile("bar.sync 1, 64;" ::: "memory");
                const bool rotate = ab * ab > tol2 * (aa * bb);  // |g_p . g_q| > sqrt(M) eps ||g_p|| ||g_q||
                if (rotate) {
                    // The rotation that makes the two columns orthogonal has tan(2 theta) = 2 ab / (bb - aa).  With
                    // d = bb - aa, r = 1/sqrt(d^2 + 4 ab^2):  cos(2 theta) = |d| r,  cos^2(theta) = x = (1 + |d| r)/2,
                    // cs = sqrt(x) = x rsqrt(x),  sn = sign(d) ab r / cs = sign(d) ab r rsqrt(x),  t = sn / cs = sn rsqrt(x)
                    // -- the smaller-angle root, same as t = sign(zeta)/(|zeta| + sqrt(1 + zeta^2)), zeta = d/(2 ab), with
                    // two dependent reciprocal square roots and no division on the chain.
                    const double d = bb - aa;
                    const double r = fast_rsqrt_pos(fma(d, d, 4.0 * ab * ab));
                    const double xx = fma(0.5 * fabs(d), r, 0.5);
                    const double rs = fast_rsqrt_pos(xx);
                    const double cs = xx * rs;
                    const double sn = ((d < 0.0) ? -ab : ab) * r * rs;
                    const double tt = sn * rs;
#pragma unroll
                    for (int e = 0; e < E2; ++e) {
                        const double2 xe = x[e], ye = y[e];
                        x[e].x = cs * xe.x - sn * ye.x; x[e].y = cs * xe.y - sn * ye.y;
                        y[e].x = sn * xe.x + cs * ye.x; y[e].y = sn * xe.y + cs * ye.y;
                    }
                    aa = fma(-tt, ab, aa);
                    bb = fma(tt, ab, bb);
                    ++nrot;
                }
                // where do the two columns sit next round?  top[t] -> top[t+1] (same slot) unless it is the
                // CTA's last top seat; bot[t] -> bot[t-1] (same slot) unless it is the CTA's first bottom seat.
                const bool top_fixed = (cr == 0 && t == 0);
                const bool top_leaves = (t == h_loc - 1) && !top_fixed;
                const bool bot_leaves = (t == 0);
                if (top_leaves) {
                    if (has_right) {  // straight from registers into the right neighbour's top spare
                        const int dslot = T0 + wrap(head_t + RT - 1, RT);
                        const uint32_t rcta = (uint32_t)(cr + 1);
                        const uint32_t rbar = mapa_shared(mbar_u32 + 8u * par, rcta);
                        const uint32_t base = mapa_shared(cols_u32 + (uint32_t)(dslot * Ms * 8), rcta) + 16u * lane;
#pragma unroll
                        for (int e = 0; e < E2; ++e) st_async_v2f64(base + 512u * e, x[e], rbar);
                        if (lane == 0) {
                            st_async_s32(mapa_shared(ids_u32 + 4u * dslot, rcta), idp, rbar);
                            st_async_f64(mapa_shared(nrm2_u32 + 8u * dslot, rcta), aa, rbar);
                        }
                    } else {          // last CTA: the column turns the corner into this CTA's bottom spare
                        const int dslot = B0 + wrap(head_b + h_loc, RT);
                        const uint32_t base = cols_u32 + (uint32_t)(dslot * Ms * 8) + 16u * lane;
#pragma unroll
                        for (int e = 0; e < E2; ++e) sts128(base + 512u * e, x[e]);
                        if (lane == 0) { ids[dslot] = idp; nrm2[dslot] = aa; }
                    }
                } else {
                    if (rotate) {
#pragma unroll
                        for (int e = 0; e < E2; ++e) sts128(ap + 512u * e, x[e]);
                    }
                    if (lane == 0 && (rotate || rnd == 0)) nrm2[sp] = aa;
                }
                if (bot_leaves) {
                    if (has_left) {   // straight from registers into the left neighbour's bottom spare
                        const int dslot = B0 + wrap(head_b + h_loc, RT);
                        const uint32_t rcta = (uint32_t)(cr - 1);
                        const uint32_t rbar = mapa_shared(mbar_u32 + 16u + 8u * par, rcta);
                        const uint32_t base = mapa_shared(cols_u32 + (uint32_t)(dslot * Ms * 8), rcta) + 16u * lane;
#pragma unroll
                        for (int e = 0; e < E2; ++e) st_async_v2f64(base + 512u * e, y[e], rbar);
                        if (lane == 0) {
                            st_async_s32(mapa_shared(ids_u32 + 4u * dslot, rcta), idq, rbar);
                            st_async_f64(mapa_shared(nrm2_u32 + 8u * dslot, rcta), bb, rbar);
                        }
                    } else {          // CTA 0: the column turns the corner into this CTA's top spare
                        const int dslot = T0 + wrap(head_t0 + RT0 - 1, RT0);
                        const uint32_t base = cols_u32 + (uint32_t)(dslot * Ms * 8) + 16u * lane;
#pragma unroll
                        for (int e = 0; e < E2; ++e) sts128(base + 512u * e, y[e]);
                        if (lane == 0) { ids[dslot] = idq; nrm2[dslot] = bb; }
                    }
                } else {
                    if (rotate) {
#pragma unroll
                        for (int e = 0; e < E2; ++e) sts128(aq + 512u * e, y[e]);
                    }
                    if (lane == 0 && (rotate || rnd == 0)) nrm2[sq] = bb;
                }
            }
            if (rnd == nrounds - 1 && lane == 0 && nrot) atomicAdd(rot + sweep, nrot);
            // The boundary columns are already on their way (sent as soon as they were rotated, so the DSMEM latency
            // hides under the other pairs).  The CTA barrier orders this round's local writes before next round's
            // reads; then wait for the two incoming columns of this round.  Point to point: nobody waits for CTAs
            // it does not exchange with.
            __syncthreads();
            if (CS > 1) {
                const uint32_t ph = (rcount >> 1) & 1u;
                if (tid == 64) {
                    if (has_left) mbar_expect_tx(mbar_u32 + 8u * par, col_tx);
                    if (has_right) mbar_expect_tx(mbar_u32 + 16u + 8u * par, col_tx);
                }
                if (has_left) mbar_wait(mbar_u32 + 8u * par, ph);
                if (has_right) mbar_wait(mbar_u32 + 16u + 8u * par, ph);
                if (rnd == nrounds - 1) cluster_sync_all();  // once per sweep: every CTA's rotation count is in
            }
            ++rcount;
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
        const double* gc = cols + (size_t)slot * Ms;
        double ss = 0.0;
        for (int r = lane; r < M; r += 32) ss = fma(gc[r], gc[r], ss);
        ss = warp_sum(ss);
        if (lane == 0 && cid < M) nrm_s[cid] = sqrt(ss);
    }
    __threadfence();
    if (CS > 1) cluster_sync_all(); else __syncthreads();
    for (int c = tid; c < M; c += NT) nrm[c] = __ldcg(nrm_s + c);
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
    for (int q = warp; q < 2 * h_loc; q += NW) {
        const int slot = q < h_loc ? slot_top(q) : slot_bot(q - h_loc);
        const int cid = ids[slot];
        if (cid >= M) continue;
        const int j = rank[cid] - off;
        if (j < 0 || j >= m) continue;
        const double nv = nrm[cid];
        const double inv = 1.0 / nv;
        const double* gc = cols + (size_t)slot * Ms;
        double* v = V + (size_t)(g0 + j) * N + lo;
        for (int r = lane; r < M; r += 32) v[r] = gc[r] * inv;
        if (lane == 0) eps[g0 + j] = nv - sigma;
    }
}

}  // namespace pfsm
