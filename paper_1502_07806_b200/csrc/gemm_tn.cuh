// gemm_tn.cuh -- FP64 tensor-core (DMMA) GEMM  C = epilogue(X * Y^T)  for sm_100a.
//
// The dense contractions of the PFSM path (Eq. 11: "a sequence of matrix-vector
// products"; all N vectors side by side make them N x N x N products) all have the same shape once
// the symmetric A is read as its own transpose:
//      C[i][j] = sum_k X[i][k] * Y[j][k]           X, Y row-major with K contiguous ("TN")
// where a "row" of the row-major view is a column of the caller's column-major matrix (row i of
// V = eigenvector i).  The same kernel serves the folded-spectrum products (Y = A), the Gram matrix
// (Y = X = V), the Cholesky panel / trailing updates and the triangular solve (Y = a panel of L).
//
// Blackwell notes.  tcgen05.mma has no FP64 kind, so the FP64 tensor primitive on sm_100a is the
// warp-level mma.sync m8n8k4 (SASS DMMA.8x8x4).  Operand tiles are staged by TMA
// (cp.async.bulk.tensor.2d, SWIZZLE_128B) through a multi-stage mbarrier full/empty pipeline filled
// by one elected lane; 8 warps each own a 64 x 32 accumulator tile (64 FP64 accumulators per
// thread) of the CTA's 128 x 128 tile.  256 threads x <=255 registers fill the register file, so
// there is no separate producer warp (a 9th warp would cap every thread at 168 registers).
//
// Shared-memory tile: 128 rows x 16 doubles (128 B per row), 16-byte chunk c of row r stored at
// chunk c ^ (r & 7) (TMA SWIZZLE_128B).  A thread (g = lane>>2, t = lane&3) reads, for k-half h,
// the 16-byte chunk (2t + h) of row g of each 8-row group: the 8 lanes of every quarter-warp hit 8
// distinct chunks -> conflict-free LDS.128.  The two doubles of that chunk are k = 4t + 2h + {0,1},
// so DMMA k-step s = 2h + e of a 16-wide k-block contracts over k in {s, 4+s, 8+s, 12+s}: a
// permutation of k applied identically to both operands, which leaves the sum unchanged.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace pfsm {

constexpr int BM = 128, BN = 128, BK = 16;
constexpr int GEMM_STAGES = 6;
constexpr int GEMM_CONSUMER_WARPS = 8;
constexpr int GEMM_THREADS = GEMM_CONSUMER_WARPS * 32;       // 256 threads x 255 registers = the whole file
constexpr int GEMM_PREFETCH = GEMM_STAGES - 2;               // k-blocks in flight ahead of the math
constexpr int TILE_BYTES = BM * BK * 8;                       // 16 KiB per operand per stage
constexpr int GEMM_MAX_PEERS = 7;                              // other ranks of one NVSwitch node (8 GPUs)
constexpr int GEMM_SMEM = GEMM_STAGES * 2 * TILE_BYTES + 1024 /*align*/ + 256 /*barriers*/;

enum Epilogue : int {
    EPI_PLAIN = 0,   // C = acc
    EPI_SHIFT = 1,   // C = acc - eps[i] * E1[i][j]                      (W = A V - V diag(eps))
    EPI_UPDATE = 2,  // C = E2[i][j] - alpha * (acc - eps[i] * E1[i][j])  (V <- V - alpha (A W - W diag(eps)))
    EPI_SUB = 3,     // C = C - acc                                       (trailing update)
    EPI_JSTEP = 4,   // C = E2[i][j] - (acc - E1[i][j]) * eps[j]           (Eq. 14: Z <- Z - D^-1 (B Z - A), eps = 1/diag(B) per COLUMN)
};

struct GemmParams {
    // region of C (row-major view, leading dimension ldc), origin (cr0, cc0), size mr x nc
    double* C;
    int64_t ldc;
    int32_t cr0, cc0, mr, nc;
    // operand coordinates: X rows start at xr0, Y rows at yr0; k runs over [0, klen) with column
    // offsets xk0 / yk0 into X / Y
    int32_t xr0, yr0, xk0, yk0, klen;
    // optional per-row-tile k-range {begin, end} (multiples of BK), overrides [0, klen)
    const int2* krange;
    // lower != 0: only tiles (tr, tc) with tr >= tc are computed (1: column by column; 2: row by row, ntr == ntc)
    int32_t lower;
    int32_t ntr, ntc;
    // epilogue operands, same coordinates as C
    const double* E1;
    int64_t ld1;
    const double* E2;
    int64_t ld2;
    const double* eps;  // indexed by absolute C row (SHIFT, UPDATE) or absolute C column (JSTEP)
    double alpha;
    // Chained launches (programmatic dependent launch, see launch_gemm): this kernel's operand X and its epilogue
    // operands are the previous kernel's output.  A tile of row block tr starts once wait_cnt[tr] == wait_target
    // (all tiles of that row block of the previous kernel have stored), and bumps signal_cnt[tr] after its own stores.
    const int32_t* wait_cnt;
    int32_t wait_target;
    int32_t* signal_cnt;
    // Batch of independent products in one launch (the per-slice trailing updates of the blocked tridiagonalization):
    // grid = nbatch * tiles_per_batch; batch b shifts the X / Y / C row origins by b * bxs / b * bys / b * bcs rows of the
    // same tensor maps (the slices' matrices are stacked row-wise).  nbatch <= 1: a single product.
    int32_t nbatch, tiles_per_batch, bxs, bys, bcs;
    // Fused compute + all-gather (gemm_tn_kernel<EPI, true> only; the sharded solve): every C tile is also
    // stored, at the same coordinates, into the buffers of npeer other ranks -- peer device memory mapped through CUDA IPC
    // (NVLink / NVSwitch P2P stores), so the exchange the paper does with MPI_Allgatherv rides on the
    // product's own epilogue, tile by tile, instead of following it as a separate collective.
    double* peerC[GEMM_MAX_PEERS];
    int32_t npeer;
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int32_t c0, int32_t c1,
                                            uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(
            dst),
        "l"(map), "r"(bar), "r"(c0), "r"(c1)
        : "memory");
}
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}
__device__ __forceinline__ double2 lds128(uint32_t addr) {
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}

// linear tile index -> (tr, tc).  Full: groups of 8 row-tiles, column-major inside a group, so that
// the ~148 co-resident CTAs share operand tiles in L2.  Lower: column-major over tiles with tr >= tc.
__device__ __forceinline__ bool tile_coords(const GemmParams& p, int32_t idx, int32_t& tr, int32_t& tc) {
    if (!p.lower) {
        constexpr int GM = 8;
        const int32_t per_group = GM * p.ntc;
        const int32_t grp = idx / per_group;
        const int32_t first = grp * GM;
        const int32_t gsz = min(GM, p.ntr - first);
        const int32_t rem = idx - grp * per_group;
        tr = first + rem % gsz;
        tc = rem / gsz;
        return tr < p.ntr && tc < p.ntc;
    }
    if (p.lower == 2) {
        // square region, row by row: row tr holds columns 0..tr, prefix(tr) = tr (tr + 1) / 2.  Early tiles only touch
        // early row blocks, which is what a chained launch (wait_cnt) needs.
        int32_t r = (int32_t)((sqrt(8.0 * (double)idx + 1.0) - 1.0) * 0.5);
        r = max(0, min(r, p.ntr - 1));
        while (r > 0 && (int64_t)r * (r + 1) / 2 > idx) --r;
        while ((int64_t)(r + 1) * (r + 2) / 2 <= idx) ++r;
        tr = r;
        tc = (int32_t)(idx - (int64_t)r * (r + 1) / 2);
        return tr < p.ntr;
    }
    // column tc holds rows tc..ntr-1: count ntr - tc; prefix(tc) = tc*ntr - tc(tc-1)/2
    const double n = (double)p.ntr + 0.5;
    int32_t c = (int32_t)(n - sqrt(n * n - 2.0 * (double)idx));
    c = max(0, min(c, p.ntc - 1));
    auto prefix = [&](int32_t t) { return (int64_t)t * p.ntr - (int64_t)t * (t - 1) / 2; };
    while (c > 0 && prefix(c) > idx) --c;
    while (c + 1 < p.ntc && prefix(c + 1) <= idx) ++c;
    tc = c;
    tr = c + (int32_t)(idx - prefix(c));
    return tr < p.ntr;
}

inline int64_t gemm_num_tiles(int32_t ntr, int32_t ntc, int lower) {
    if (!lower) return (int64_t)ntr * ntc;
    if (lower == 2) return (int64_t)ntr * (ntr + 1) / 2;
    int64_t t = 0;
    for (int c = 0; c < ntc; ++c) t += (ntr - c > 0 ? ntr - c : 0);
    return t;
}

template <int EPI, bool PEER = false>
__global__ void __launch_bounds__(GEMM_THREADS, 1)
gemm_tn_kernel(const __grid_constant__ CUtensorMap mapX, const __grid_constant__ CUtensorMap mapY,
               const __grid_constant__ CUtensorMap mapC, const GemmParams p) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;  // SWIZZLE_128B needs 1024-B alignment
    const uint32_t bar_base = smem_base + GEMM_STAGES * 2 * TILE_BYTES;
    // full[s] at bar_base + 8 s, empty[s] at bar_base + 8 (STAGES + s)

    // lets a kernel launched with programmatic stream serialization become resident while this grid's last wave runs
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

    int32_t tr, tc;
    int32_t bidx = (int32_t)blockIdx.x, batch = 0;
    if (p.nbatch > 1) {
        batch = bidx / p.tiles_per_batch;
        bidx -= batch * p.tiles_per_batch;
    }
    if (!tile_coords(p, bidx, tr, tc)) return;
    const int32_t cr0 = p.cr0 + batch * p.bcs;  // C row origin of this batch entry

    int32_t kb0 = 0, nk = (p.klen + BK - 1) / BK;
    if (p.krange) {
        const int2 kr = p.krange[tr];
        kb0 = kr.x / BK;
        nk = (kr.y - kr.x + BK - 1) / BK;
    }

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < GEMM_STAGES; ++s) {
            mbar_init(bar_base + 8 * s, 1);
            mbar_init(bar_base + 8 * (GEMM_STAGES + s), GEMM_CONSUMER_WARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        if (p.wait_cnt) {
            // The producer grid is resident or finished (it triggered the dependent launch from every CTA), so this
            // spin cannot starve it.  acquire + bar.sync order every thread's later loads, the proxy fence the TMA reads.
            // a lower-triangular product X X^T also reads row block tc of the previous output (tc <= tr)
            for (int32_t rb = p.lower ? tc : tr; rb <= tr; rb += max(1, tr - tc)) {
                const int32_t* c = p.wait_cnt + rb;
                int32_t seen;
                for (;;) {
                    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(seen) : "l"(c) : "memory");
                    if (seen >= p.wait_target) break;
                    __nanosleep(256);
                }
            }
            asm volatile("fence.proxy.async.global;" ::: "memory");
        }
    }
    __syncthreads();

    // ===== TMA producer = lane 0 of warp 0, interleaved with its math.  At the top of iteration kb it
    // refills the stage that every warp finished two iterations ago (k-block kb + PREFETCH), so the
    // wait on that stage's empty barrier almost never blocks and 4 k-blocks stay in flight. =====
    const int32_t xrow = p.xr0 + batch * p.bxs + tr * BM, yrow = p.yr0 + batch * p.bys + tc * BN;
    auto issue = [&](int32_t j) {
        const int s = j % GEMM_STAGES;
        if (j >= GEMM_STAGES) mbar_wait(bar_base + 8 * (GEMM_STAGES + s), ((j / GEMM_STAGES) - 1) & 1);
        const uint32_t full = bar_base + 8 * s;
        mbar_expect_tx(full, 2 * TILE_BYTES);
        const int32_t k = (kb0 + j) * BK;
        tma_load_2d(smem_base + s * 2 * TILE_BYTES, &mapX, p.xk0 + k, xrow, full);
        tma_load_2d(smem_base + s * 2 * TILE_BYTES + TILE_BYTES, &mapY, p.yk0 + k, yrow, full);
    };
    if (threadIdx.x == 0) {
        const int32_t npre = nk < GEMM_PREFETCH ? nk : GEMM_PREFETCH;
        for (int32_t j = 0; j < npre; ++j) issue(j);
    }
    if ((EPI == EPI_SUB || EPI == EPI_UPDATE || EPI == EPI_JSTEP) && threadIdx.x == 32) {
        // the epilogue reads the C tile: pull it from HBM into L2 now, under the main loop (mapC describes C)
#pragma unroll
        for (int j = 0; j < BN / BK; ++j)
            asm volatile("cp.async.bulk.prefetch.tensor.2d.L2.global.tile [%0, {%1, %2}];" ::"l"(&mapC),
                         "r"(p.cc0 + tc * BN + j * BK), "r"(cr0 + tr * BM)
                         : "memory");
    }

    // ===== consumers: warp (wr, wc) of a 2 x 4 grid owns rows [64 wr, +64) x cols [32 wc, +32) =====
    const int wr = warp >> 2, wc = warp & 3;
    const int g = lane >> 2, t = lane & 3;
    double acc[8][4][2];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    // byte offsets inside a tile for the two k-halves (row g of a group, swizzled chunk)
    const uint32_t off_h0 = (uint32_t)(g * 128 + (((2 * t + 0) ^ g) << 4));
    const uint32_t off_h1 = (uint32_t)(g * 128 + (((2 * t + 1) ^ g) << 4));
    const uint32_t a_warp = (uint32_t)(wr * 64 * 128);
    const uint32_t b_warp = (uint32_t)(TILE_BYTES + wc * 32 * 128);

    for (int32_t kb = 0; kb < nk; ++kb) {
        if (threadIdx.x == 0 && kb + GEMM_PREFETCH < nk) issue(kb + GEMM_PREFETCH);
        __syncwarp();
        const int s = kb % GEMM_STAGES;
        mbar_wait(bar_base + 8 * s, (kb / GEMM_STAGES) & 1);
        const uint32_t st = smem_base + s * 2 * TILE_BYTES;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const uint32_t off = h ? off_h1 : off_h0;
            double2 a[8], b[4];
#pragma unroll
            for (int i = 0; i < 8; ++i) a[i] = lds128(st + a_warp + i * 1024 + off);
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = lds128(st + b_warp + j * 1024 + off);
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma884(acc[i][j][0], acc[i][j][1], a[i].x, b[j].x);
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) dmma884(acc[i][j][0], acc[i][j][1], a[i].y, b[j].y);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_base + 8 * (GEMM_STAGES + s));
    }

    // chained launches: publish this tile (every thread's stores, for generic and TMA readers) and count it
    auto signal_done = [&]() {
        if (!p.signal_cnt) return;
        __threadfence();
        asm volatile("fence.proxy.async.global;" ::: "memory");
        __syncthreads();
        if (threadIdx.x == 0) asm volatile("red.release.gpu.global.add.s32 [%0], 1;" ::"l"(p.signal_cnt + tr) : "memory");
    };

    // ===== epilogue: thread owns C[row0 + 8 i + g][col0 + 8 j + 2 t + {0,1}] =====
    const int32_t row0 = tr * BM + wr * 64, col0 = tc * BN + wc * 32;
    if (EPI != EPI_PLAIN && (tr + 1) * BM <= p.mr && (tc + 1) * BN <= p.nc) {
        // Interior tile: no bounds checks, and the epilogue operands are fetched 16 x 16 bytes at a time before
        // they are used -- 2 memory round trips per thread instead of 32 dependent load -> store chains.
        const int64_t base = ((int64_t)cr0 + row0 + g) * p.ldc + p.cc0 + col0 + 2 * t;  // ldc == ld1 == ld2 here
        double2 dj[4];
        if (EPI == EPI_JSTEP) {
#pragma unroll
            for (int j = 0; j < 4; ++j) dj[j] = *reinterpret_cast<const double2*>(p.eps + p.cc0 + col0 + 8 * j + 2 * t);
        }
#pragma unroll
        for (int ib = 0; ib < 8; ib += 4) {
            double2 u[4][4], w[4][4];
            double e[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int64_t o = base + (int64_t)(8 * (ib + i)) * p.ldc;
                if (EPI == EPI_SHIFT || EPI == EPI_UPDATE) e[i] = p.eps[(int64_t)cr0 + row0 + 8 * (ib + i) + g];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    if (EPI == EPI_SHIFT || EPI == EPI_UPDATE || EPI == EPI_JSTEP)
                        u[i][j] = __ldcg(reinterpret_cast<const double2*>(p.E1 + o + 8 * j));
                    if (EPI == EPI_UPDATE || EPI == EPI_JSTEP) w[i][j] = __ldcg(reinterpret_cast<const double2*>(p.E2 + o + 8 * j));
                    if (EPI == EPI_SUB) w[i][j] = *reinterpret_cast<const double2*>(p.C + o + 8 * j);
                }
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int64_t o = base + (int64_t)(8 * (ib + i)) * p.ldc;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    double v0 = acc[ib + i][j][0], v1 = acc[ib + i][j][1];
                    if (EPI == EPI_SHIFT) {
                        v0 -= e[i] * u[i][j].x;
                        v1 -= e[i] * u[i][j].y;
                    } else if (EPI == EPI_UPDATE) {
                        v0 = w[i][j].x - p.alpha * (v0 - e[i] * u[i][j].x);
                        v1 = w[i][j].y - p.alpha * (v1 - e[i] * u[i][j].y);
                    } else if (EPI == EPI_JSTEP) {
                        v0 = w[i][j].x - (v0 - u[i][j].x) * dj[j].x;
                        v1 = w[i][j].y - (v1 - u[i][j].y) * dj[j].y;
                    } else {
                        v0 = w[i][j].x - v0;
                        v1 = w[i][j].y - v1;
                    }
                    *reinterpret_cast<double2*>(p.C + o + 8 * j) = make_double2(v0, v1);
                    if (PEER) {
                        for (int q = 0; q < p.npeer; ++q) *reinterpret_cast<double2*>(p.peerC[q] + o + 8 * j) = make_double2(v0, v1);
                    }
                }
            }
        }
        if (PEER) __threadfence_system();  // peer stores: visible to the other devices before this grid is seen complete
        signal_done();
        return;
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int32_t r = row0 + 8 * i + g;
        if (r >= p.mr) continue;
        const int64_t ar = (int64_t)cr0 + r;
        double e = 0.0;
        if (EPI == EPI_SHIFT || EPI == EPI_UPDATE) e = p.eps[ar];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int32_t c = col0 + 8 * j + 2 * t;
            if (c >= p.nc) continue;
            const int64_t ac = (int64_t)p.cc0 + c;
            double v0 = acc[i][j][0], v1 = acc[i][j][1];
            const bool pair = (c + 1 < p.nc);
            double* cp = p.C + ar * p.ldc + ac;
            if (EPI == EPI_SHIFT) {
                const double* e1 = p.E1 + ar * p.ld1 + ac;
                if (pair) {
                    const double2 x = __ldcg(reinterpret_cast<const double2*>(e1));
                    v0 -= e * x.x;
                    v1 -= e * x.y;
                } else
                    v0 -= e * __ldcg(e1);
            } else if (EPI == EPI_UPDATE) {
                const double* e1 = p.E1 + ar * p.ld1 + ac;
                const double* e2 = p.E2 + ar * p.ld2 + ac;
                if (pair) {
                    const double2 x = __ldcg(reinterpret_cast<const double2*>(e1));
                    const double2 y = __ldcg(reinterpret_cast<const double2*>(e2));
                    v0 = y.x - p.alpha * (v0 - e * x.x);
                    v1 = y.y - p.alpha * (v1 - e * x.y);
                } else
                    v0 = __ldcg(e2) - p.alpha * (v0 - e * __ldcg(e1));
            } else if (EPI == EPI_JSTEP) {
                const double* e1 = p.E1 + ar * p.ld1 + ac;
                const double* e2 = p.E2 + ar * p.ld2 + ac;
                v0 = e2[0] - (v0 - e1[0]) * p.eps[ac];
                if (pair) v1 = e2[1] - (v1 - e1[1]) * p.eps[ac + 1];
            } else if (EPI == EPI_SUB) {
                if (pair) {
                    const double2 y = *reinterpret_cast<const double2*>(cp);
                    v0 = y.x - v0;
                    v1 = y.y - v1;
                } else
                    v0 = cp[0] - v0;
            }
            if (pair)
                *reinterpret_cast<double2*>(cp) = make_double2(v0, v1);
            else
                cp[0] = v0;
            if (PEER) {
                for (int q = 0; q < p.npeer; ++q) {
                    double* pp = p.peerC[q] + ar * p.ldc + ac;
                    if (pair)
                        *reinterpret_cast<double2*>(pp) = make_double2(v0, v1);
                    else
                        pp[0] = v0;
                }
            }
        }
    }
    if (PEER) __threadfence_system();
    signal_done();
}

}  // namespace pfsm
