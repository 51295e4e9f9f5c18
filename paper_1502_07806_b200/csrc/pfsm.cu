// pfsm.cu -- C-ABI boundary (include/pfsm.h) and step orchestration of one PFSM solve on sm_100a.
// Steps and citations: see include/pfsm.h.  All compute runs in the kernels of gemm_tn.cuh and
// kernels.cuh on the caller's stream; the host only validates arguments, encodes TMA descriptors
// and enqueues launches.  There is no CPU fallback.
#include "../../include/pfsm.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <climits>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <vector>

#include "gemm_tn.cuh"
#include "kernels.cuh"
#include "jacobi_smem.cuh"
#include "jacobi_wide.cuh"
#include "tridiag_eig.cuh"
#include "sytrd_blocked.cuh"

namespace pfsm {

#define PFSM_CUDA(call)                                              \
    do {                                                             \
        cudaError_t e__ = (call);                                    \
        if (e__ != cudaSuccess) return PFSM_CUDA_ERROR_BASE + (int)e__; \
    } while (0)

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

// 2-D FP64 tensor map over a row-major (rows x cols, leading dimension ld) matrix; box = 128 rows x 16
// doubles (one 128-byte swizzle span); out-of-bounds elements read as zero.
static int make_map(CUtensorMap* map, const double* base, int64_t rows, int64_t cols, int64_t ld) {
    EncodeTiledFn fn = get_encode_fn();
    if (!fn) return PFSM_CUDA_ERROR_BASE + (int)cudaErrorNotSupported;
    cuuint64_t gdim[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
    cuuint64_t gstr[1] = {(cuuint64_t)ld * 8};
    cuuint32_t box[2] = {(cuuint32_t)BK, (cuuint32_t)BM};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void*)base, gdim, gstr, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? 0 : PFSM_CUDA_ERROR_BASE + (int)cudaErrorInvalidValue;
}

}  // namespace pfsm

using namespace pfsm;

// ---- Scratch of the allocation-free entry point pfsm_rayleigh_noalloc (below): T = V A of step 5, N <= 1024.
// 8 MiB of device memory on every GPU that loads the library, held until the process exits.  In HOST code this name is a
// host-side stand-in, not a device address: the address kernels and tensor maps use comes from cudaGetSymbolAddress, once
// per device, with that device current (noalloc_scratch_ptr).
#define PFSM_NOALLOC_MAX_N 1024
static __device__ __align__(256) double pfsm_noalloc_scratch[(size_t)PFSM_NOALLOC_MAX_N * PFSM_NOALLOC_MAX_N];

static int noalloc_scratch_ptr(double** out) {
    constexpr int MAXDEV = 64;
    static double* addr[MAXDEV] = {nullptr};
    static std::mutex mu;
    int dev = -1;
    PFSM_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAXDEV) return PFSM_CUDA_ERROR_BASE + (int)cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        void* p = nullptr;
        PFSM_CUDA(cudaGetSymbolAddress(&p, pfsm_noalloc_scratch));  // the CURRENT device's instance of the array
        addr[dev] = (double*)p;
    }
    *out = addr[dev];
    return 0;
}

struct pfsm_ctx {
    int64_t N;
    int64_t ld;               // leading dimension of every internal N x N matrix: N rounded up to even (TMA needs a 16-byte row pitch)
    double* padA = nullptr;   // odd N: the caller's matrices (ld = N) are staged through these (ld = N + 1)
    double* padB = nullptr;
    double* padV = nullptr;
    double* Ub = nullptr;     // pfsm_solve_warm: eigenvectors of the rotated problem
    int32_t P, window, iters, m, M;
    double alpha;
    int device;
    // device workspace
    double* W = nullptr;      // N x N   : W of step 3, T of step 5
    double* S = nullptr;      // 2N x N  : stacked [G ; V^T] of step 4
    double* O = nullptr;      // 2N x N  : stacked [L ; V^T R^-1]
    double* Dinv = nullptr;   // nblk x 128 x 128 : inverses of L's diagonal blocks
    double* Gws = nullptr;    // P x M x M : Jacobi workspace
    double* eps = nullptr;    // N shifts
    double* resid = nullptr;  // N residual norms
    int* rotcnt = nullptr;    // P x JACOBI_MAX_SWEEPS rotation counters of step 2
    unsigned int* jw_bar = nullptr;  // grid-barrier counter of the wide-window Jacobi (M > 512)
    double* nrm_g = nullptr;  // P x (M + 16): final column norms of the shared-memory Jacobi
    bool jac_wide = false;             // persistent-grid Jacobi (jacobi_wide.cuh): option step2_route = 3, at any M
    bool tridiag = false;              // tridiagonalization route (tridiag_eig.cuh): default for M >= 16, step2_route = 2 at any M
    TriWs tri{};                       // its workspace
    SbWs sbw{};                        // workspace of the blocked tridiagonalization (sytrd_blocked.cuh), allocated on first use
    CUtensorMap mapG, mapVW, mapWV;    //   its tensor maps: the stacked submatrices (P M x M) and panel operands (P M x 2 NB)
    int jac_cs = 0, jac_hloc = 0;  // cluster size / seats per CTA of the shared-memory Jacobi (0 = L2 kernel)
    double* gdiag = nullptr;  // N: diag(V^T V) before the factorization (breakdown threshold)
    int32_t* slice_tab = nullptr;  // g0[P], lo[P], off[P], cnt[P]
    std::vector<int32_t> tab_host;  // the same table on the host
    int2* krange = nullptr;        // per 128-row tile k-range of the first product
    unsigned long long* info = nullptr;
    double* Ap = nullptr;       // generalized variant: A' = L^-1 A L^-T
    double* LT = nullptr;       //   L^T (S = L L^T)
    double* DinvT = nullptr;    //   transposed inverses of L's diagonal blocks
    CUtensorMap mapAp, mapLT, mapDT;
    double* A_stage = nullptr;  // host-buffer path
    double* V_stage = nullptr;
    double* lam_stage = nullptr;
    size_t bytes = 0;
    int32_t nblk;
    CUtensorMap mapW, mapS, mapO, mapD;
    bool timing = false;
    cudaEvent_t ev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    bool ev_valid = false;
    bool keep_info = false;
    cudaStream_t side = nullptr;       // high-priority stream of the Cholesky look-ahead
    cudaEvent_t ev_chain = nullptr, ev_rest = nullptr, ev_fork = nullptr;
    bool lookahead = true;
    bool chain = true;                 // step 3: consecutive GEMMs overlap their last waves (row-block counters + PDL)
    int32_t* chain_cnt = nullptr;      // [2 * iters][ceil(N / BM)] tiles stored per row block of each step-3 GEMM
    int32_t cholqr_passes = 1;         // 2 = CholeskyQR2 (re-orthonormalize once; reading R10)
    bool jac_half = false;             // shared-memory Jacobi with 512-thread CTAs, two per SM (jacobi_smem.cuh)
    int32_t sh_rank = 0, sh_world = 1;  // sharded solve: this handle works on rows [sh_rank, sh_rank+1) * N / sh_world
    // peer-write mode of the sharded solve (pfsm_set_shard_peers): the other ranks' copies of V, buffer 0 (G), buffer 1
    // (V^T R^-1), lambda and the residuals, mapped into this process; npeer = 0: the caller all-gathers instead
    double* peer_buf[5][GEMM_MAX_PEERS] = {};
    int32_t npeer = 0;
    bool gemm_attr_peer[5] = {false, false, false, false, false};
    // per-handle launch state (function attributes are per device/context, so nothing here is a process-wide static)
    int sms = 0;                       // multiprocessors of h->device
    bool gemm_attr[5] = {false, false, false, false, false};  // MaxDynamicSharedMemorySize set for gemm_tn_kernel<EPI>
    bool pdl_ok = true;                // cleared if the driver refuses programmatic stream serialization
    bool chol_attr = false;
    // options (pfsm_set_option; defaults = the product path)
    int32_t opt_route = 0;             // step2_route: 0 auto, 1 Jacobi family (M <= 512), 2 tridiagonal, 3 persistent-grid Jacobi
    int32_t opt_jacobi_l2 = 0;         // 1: L2-resident Jacobi kernel instead of the shared-memory one
    int32_t opt_jacobi_cs = 0;         // cluster size of the shared-memory Jacobi (0 = auto)
    int32_t opt_jacobi_full = 0;       // 1: no half-CTA layout
    int32_t opt_sytrd_storage = 0;     // 0 auto, 1 full storage, 2 lower triangle
    int32_t opt_sytrd_grid = 0;        // 1: grid barrier instead of clusters for small M
    int32_t opt_chol_group = 0;        // panels per trailing update of step 4: 0 auto, 2, 4
};

// largest submatrix order: the tridiagonal route's back-transformation keeps M / 256 <= 32 doubles per thread and vector
constexpr int64_t PFSM_MAX_M = 8192;

static int dev_alloc(pfsm_ctx* h, void** p, size_t bytes) {
    PFSM_CUDA(cudaMalloc(p, bytes));
    h->bytes += bytes;
    return 0;
}

// Every entry point that enqueues work runs on the handle's device: workspace, tensor maps and function attributes
// belong to it.  A caller that switched devices gets an error instead of a launch on the wrong context.
static int check_device(const pfsm_ctx* h) {
    int dev = -1;
    PFSM_CUDA(cudaGetDevice(&dev));
    return dev == h->device ? 0 : PFSM_CUDA_ERROR_BASE + (int)cudaErrorInvalidDevice;
}

// Odd N: a caller matrix (N x N, leading dimension N) cannot be described by a tensor map (its row pitch is not a multiple
// of 16 bytes), so it is staged through an internal copy with leading dimension ld = N + 1.  Even N: used in place.
static int copy_mat(double* dst, int64_t dld, const double* src, int64_t sld, int64_t N, cudaStream_t st) {
    PFSM_CUDA(cudaMemcpy2DAsync(dst, (size_t)dld * sizeof(double), src, (size_t)sld * sizeof(double), (size_t)N * sizeof(double),
                                (size_t)N, cudaMemcpyDeviceToDevice, st));
    return 0;
}
// *use = src itself (even N) or the padded copy in *pad (allocated on first use; filled when `fill`)
static int stage_in(pfsm_ctx* h, const double* src, double** pad, double** use, cudaStream_t st, bool fill = true) {
    if (h->ld == h->N) { *use = const_cast<double*>(src); return 0; }
    int rc;
    if (!*pad && (rc = dev_alloc(h, (void**)pad, (size_t)h->N * h->ld * sizeof(double)))) return rc;
    *use = *pad;
    return fill ? copy_mat(*pad, h->ld, src, h->N, h->N, st) : 0;
}
static int stage_out(pfsm_ctx* h, const double* use, double* dst, cudaStream_t st) {
    return (use == dst) ? 0 : copy_mat(dst, h->N, use, h->ld, h->N, st);
}

// mc: tensor map of the matrix C lives in (used by the SUB / UPDATE epilogues to prefetch the C tile into L2)
template <int EPI, bool PEER = false>
// pdl: launch with programmatic stream serialization -- the grid may become resident while the previous gemm_tn_kernel
// in the stream drains its last wave; p.wait_cnt must then carry the real dependency (GemmParams).
static int launch_gemm(pfsm_ctx* h, const CUtensorMap& mx, const CUtensorMap& my, const CUtensorMap& mc, GemmParams p,
                       cudaStream_t st, bool pdl = false) {
    p.ntr = (p.mr + BM - 1) / BM;
    p.ntc = (p.nc + BN - 1) / BN;
    if (p.mr <= 0 || p.nc <= 0) return 0;
    const int64_t tiles1 = gemm_num_tiles(p.ntr, p.ntc, p.lower);
    if (tiles1 <= 0) return 0;
    p.tiles_per_batch = (int32_t)tiles1;
    const int64_t tiles = tiles1 * (p.nbatch > 1 ? p.nbatch : 1);
    bool& attr_done = PEER ? h->gemm_attr_peer[EPI] : h->gemm_attr[EPI];
    if (!attr_done) {
        PFSM_CUDA((cudaFuncSetAttribute(gemm_tn_kernel<EPI, PEER>, cudaFuncAttributeMaxDynamicSharedMemorySize, GEMM_SMEM)));
        attr_done = true;
    }
    if (pdl && h->pdl_ok) {
        cudaLaunchConfig_t cfg;
        memset(&cfg, 0, sizeof(cfg));
        cfg.gridDim = dim3((unsigned)tiles);
        cfg.blockDim = dim3(GEMM_THREADS);
        cfg.dynamicSmemBytes = GEMM_SMEM;
        cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at;
        cfg.numAttrs = 1;
        const cudaError_t e = cudaLaunchKernelEx(&cfg, gemm_tn_kernel<EPI, PEER>, mx, my, mc, p);
        if (e == cudaSuccess) return 0;
        // only "attribute not supported" falls back to plain stream order (always correct); anything else is a real error
        if (e != cudaErrorNotSupported) return PFSM_CUDA_ERROR_BASE + (int)e;
        cudaGetLastError();
        h->pdl_ok = false;
    }
    gemm_tn_kernel<EPI, PEER><<<(unsigned)tiles, GEMM_THREADS, GEMM_SMEM, st>>>(mx, my, mc, p);
    PFSM_CUDA(cudaGetLastError());
    return 0;
}

static GemmParams base_params() {
    GemmParams p;
    memset(&p, 0, sizeof(p));
    return p;
}

extern "C" { static void choose_jacobi_layout(pfsm_ctx* h); }

// workspace of the tridiagonal route of step 2 (allocated when that route is selected: at create, or by pfsm_set_option)
static int ensure_tridiag_ws(pfsm_ctx* h) {
    if (!h->tridiag || h->tri.d) return 0;
    const int64_t N = h->N, M = h->M, P = h->P;
    const size_t pm = (size_t)P * M * sizeof(double), mn = (size_t)M * h->ld;
    int rc;
#define TRYA(x) do { if ((rc = (x))) return rc; } while (0)
    TRYA(dev_alloc(h, (void**)&h->tri.d, pm));
    TRYA(dev_alloc(h, (void**)&h->tri.e, pm));
    TRYA(dev_alloc(h, (void**)&h->tri.tau, pm));
    TRYA(dev_alloc(h, (void**)&h->tri.pbuf, 2 * pm));
    TRYA(dev_alloc(h, (void**)&h->tri.vbuf, 2 * pm));
    TRYA(dev_alloc(h, (void**)&h->tri.rowbuf, pm * ((M + 31) / 32)));
    TRYA(dev_alloc(h, (void**)&h->tri.colbuf, pm * ((M + 31) / 32)));
    TRYA(dev_alloc(h, (void**)&h->tri.colk, 2 * pm));
    TRYA(dev_alloc(h, (void**)&h->tri.lam, N * sizeof(double)));
    TRYA(dev_alloc(h, (void**)&h->tri.zscale, N * sizeof(double)));
    for (int i = 0; i < 5; ++i) TRYA(dev_alloc(h, (void**)&h->tri.f[i], mn * sizeof(double)));
    TRYA(dev_alloc(h, (void**)&h->tri.piv, mn));
#undef TRYA
    return 0;
}

extern "C" {

const char* pfsm_strerror(int code) {
    if (code == 0) return "success";
    if (code < 0) {
        static const char* names[] = {"", "argument 1 invalid", "argument 2 invalid", "argument 3 invalid",
                                      "argument 4 invalid", "argument 5 invalid", "argument 6 invalid"};
        return (-code <= 6) ? names[-code] : "invalid argument";
    }
    if (code == PFSM_ERR_NOALLOC_SIZE)
        return "size not served by the allocation-free entry point (pfsm_rayleigh_noalloc: N even, 2 <= N <= 1024)";
    if (code >= PFSM_CUDA_ERROR_BASE) return cudaGetErrorString((cudaError_t)(code - PFSM_CUDA_ERROR_BASE));
    return "unknown error";
}

int pfsm_create(pfsm_handle_t* out, int64_t N, int32_t P, int32_t window, int32_t iters, double alpha) {
    if (!out) return -1;
    *out = nullptr;
    if (N < 2 || N > (1 << 30)) return -2;
    if (P < 1 || P > N) return -3;
    if (window < 0) return -4;
    if (iters < 0) return -5;
    if (!std::isfinite(alpha) || !(alpha > 0.0)) return -6;
    const int64_t m = (N + P - 1) / P;  // largest slice; all slices have N / P eigenpairs when P divides N (R14)
    const int64_t M = std::min<int64_t>(N, m + 2 * (int64_t)window);
    if (M > PFSM_MAX_M) return -4;

    pfsm_ctx* h = new pfsm_ctx();
    h->N = N; h->ld = N + (N & 1); h->P = P; h->window = window; h->iters = iters; h->alpha = alpha;
    h->m = (int32_t)m; h->M = (int32_t)M;
    h->nblk = (int32_t)((N + CHOL_NB - 1) / CHOL_NB);
    int rc = 0;
#define TRY(x) do { rc = (x); if (rc) { pfsm_destroy(h); return rc; } } while (0)
    {
        cudaError_t e = cudaGetDevice(&h->device);
        if (e != cudaSuccess) { delete h; return PFSM_CUDA_ERROR_BASE + (int)e; }
    }
    const int64_t L = h->ld;
    const size_t n2 = (size_t)N * L * sizeof(double);
    TRY(dev_alloc(h, (void**)&h->W, n2));
    TRY(dev_alloc(h, (void**)&h->S, 2 * n2));
    TRY(dev_alloc(h, (void**)&h->O, 2 * n2));
    TRY(dev_alloc(h, (void**)&h->Dinv, (size_t)h->nblk * CHOL_NB * CHOL_NB * sizeof(double)));
    TRY(dev_alloc(h, (void**)&h->Gws, (size_t)P * M * M * sizeof(double)));
    TRY(dev_alloc(h, (void**)&h->eps, N * sizeof(double)));
    TRY(dev_alloc(h, (void**)&h->resid, N * sizeof(double)));
    TRY(dev_alloc(h, (void**)&h->gdiag, N * sizeof(double)));
    TRY(dev_alloc(h, (void**)&h->rotcnt, (size_t)P * JACOBI_MAX_SWEEPS * sizeof(int)));
    TRY(dev_alloc(h, (void**)&h->nrm_g, (size_t)P * (M + 16) * sizeof(double)));
    TRY(dev_alloc(h, (void**)&h->jw_bar, sizeof(unsigned int)));
    {
        cudaError_t e = cudaDeviceGetAttribute(&h->sms, cudaDevAttrMultiProcessorCount, h->device);
        if (e != cudaSuccess) { pfsm_destroy(h); return PFSM_CUDA_ERROR_BASE + (int)e; }
    }
    choose_jacobi_layout(h);
    TRY(ensure_tridiag_ws(h));
    TRY(dev_alloc(h, (void**)&h->slice_tab, 4 * (size_t)P * sizeof(int32_t)));
    const int32_t ntr = (int32_t)((N + BM - 1) / BM);
    TRY(dev_alloc(h, (void**)&h->krange, (size_t)ntr * sizeof(int2)));
    TRY(dev_alloc(h, (void**)&h->info, sizeof(unsigned long long)));
    TRY(dev_alloc(h, (void**)&h->chain_cnt, (size_t)2 * (iters > 0 ? iters : 1) * ntr * sizeof(int32_t)));

    // step 1: slice table, and the k-range each 128-row tile of the first product needs
    std::vector<int32_t>& tab = h->tab_host;
    tab.resize(4 * (size_t)P);
    for (int32_t s = 0; s < P; ++s) {
        const int64_t g0 = ((int64_t)s * N) / P, g1 = ((int64_t)(s + 1) * N) / P;
        const int64_t lo = std::min<int64_t>(std::max<int64_t>(g0 - window, 0), N - M);
        tab[s] = (int32_t)g0;
        tab[P + s] = (int32_t)lo;
        tab[2 * (size_t)P + s] = (int32_t)(g0 - lo);
        tab[3 * (size_t)P + s] = (int32_t)(g1 - g0);
    }
    std::vector<int2> kr(ntr);
    {
        int32_t s0 = 0, s1 = 0;  // slices of the first and last row of the tile (lo is non-decreasing in s)
        for (int32_t t = 0; t < ntr; ++t) {
            const int64_t i0 = (int64_t)t * BM, i1 = std::min<int64_t>(N, i0 + BM) - 1;
            while (s0 + 1 < P && tab[s0 + 1] <= i0) ++s0;
            while (s1 + 1 < P && tab[s1 + 1] <= i1) ++s1;
            const int64_t lo0 = tab[P + s0], hi1 = tab[P + s1] + M;
            kr[t].x = (int)(lo0 / BK * BK);
            kr[t].y = (int)((hi1 + BK - 1) / BK * BK);
        }
    }
    {
        cudaError_t e = cudaMemcpy(h->slice_tab, tab.data(), tab.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemcpy(h->krange, kr.data(), kr.size() * sizeof(int2), cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemset(h->info, 0xFF, sizeof(unsigned long long));
        if (e == cudaSuccess) e = cudaMemset(h->resid, 0, N * sizeof(double));
        if (e == cudaSuccess) e = cudaMemset(h->eps, 0, N * sizeof(double));
        if (e != cudaSuccess) { pfsm_destroy(h); return PFSM_CUDA_ERROR_BASE + (int)e; }
    }
    TRY(make_map(&h->mapW, h->W, N, N, L));
    TRY(make_map(&h->mapS, h->S, 2 * N, N, L));
    TRY(make_map(&h->mapO, h->O, 2 * N, N, L));
    TRY(make_map(&h->mapD, h->Dinv, (int64_t)h->nblk * CHOL_NB, CHOL_NB, CHOL_NB));
    for (int i = 0; i < 5; ++i) {
        cudaError_t e = cudaEventCreate(&h->ev[i]);
        if (e != cudaSuccess) { pfsm_destroy(h); return PFSM_CUDA_ERROR_BASE + (int)e; }
    }
    {
        int lo_prio = 0, hi_prio = 0;
        cudaError_t e = cudaDeviceGetStreamPriorityRange(&lo_prio, &hi_prio);
        if (e == cudaSuccess) e = cudaStreamCreateWithPriority(&h->side, cudaStreamNonBlocking, hi_prio);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->ev_chain, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->ev_rest, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming);
        if (e != cudaSuccess) { pfsm_destroy(h); return PFSM_CUDA_ERROR_BASE + (int)e; }
    }
#undef TRY
    *out = h;
    return 0;
}

int pfsm_destroy(pfsm_handle_t h) {
    if (!h) return 0;
    int cur = -1;
    cudaGetDevice(&cur);
    if (cur != h->device) cudaSetDevice(h->device);
    cudaDeviceSynchronize();
    void* ptrs[] = {h->W, h->S, h->O, h->Dinv, h->Gws, h->eps, h->resid, h->gdiag, h->rotcnt, h->nrm_g, h->jw_bar, h->slice_tab, h->krange, h->info, h->chain_cnt,
                    h->A_stage, h->V_stage, h->lam_stage, h->Ap, h->LT, h->DinvT, h->padA, h->padB, h->padV, h->Ub,
                    h->tri.d, h->tri.e, h->tri.tau, h->tri.pbuf, h->tri.vbuf, h->tri.rowbuf, h->tri.colbuf, h->tri.colk, h->tri.lam, h->tri.zscale,
                    h->tri.f[0], h->tri.f[1], h->tri.f[2], h->tri.f[3], h->tri.f[4], h->tri.piv,
                    h->sbw.VW, h->sbw.WV, h->sbw.ypart, h->sbw.y, h->sbw.base, h->sbw.dots, h->sbw.yv, h->sbw.sbar};
    for (void* p : ptrs)
        if (p) cudaFree(p);
    for (int i = 0; i < 5; ++i)
        if (h->ev[i]) cudaEventDestroy(h->ev[i]);
    if (h->ev_chain) cudaEventDestroy(h->ev_chain);
    if (h->ev_rest) cudaEventDestroy(h->ev_rest);
    if (h->ev_fork) cudaEventDestroy(h->ev_fork);
    if (h->side) cudaStreamDestroy(h->side);
    if (cur >= 0 && cur != h->device) cudaSetDevice(cur);
    delete h;
    return 0;
}

static int jacobi_cluster_size(const pfsm_ctx* h) {
    // CTAs per slice: as many as fit the chip (148 SMs / P slices) but no more warps than column pairs
    const int npairs = (h->M + 1) / 2;
    int cs = 1;
    const int nw = jacobi_l2_threads(h->M > 256 ? 16 : (h->M > 128 ? 8 : 4)) / 32;  // warps per CTA
    while (cs < 8 && (2 * cs) * h->P <= h->sms && cs * nw < npairs) cs *= 2;
    return cs;
}

extern "C++" {
template <int EPL>
static int launch_jacobi_t(pfsm_ctx* h, const double* A, double* V, cudaStream_t st, int32_t s0, int32_t ns) {
    SliceTable tab{h->slice_tab, h->slice_tab + h->P, h->slice_tab + 2 * (size_t)h->P, h->slice_tab + 3 * (size_t)h->P};
    const int cs = jacobi_cluster_size(h);
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3((unsigned)(ns * cs));
    cfg.blockDim = dim3(jacobi_l2_threads(EPL));
    cfg.dynamicSmemBytes = (size_t)h->M * (sizeof(double) + sizeof(int));
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)cs;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    PFSM_CUDA(cudaLaunchKernelEx(&cfg, jacobi_batched_kernel<EPL>, A, h->ld, h->M, tab, h->Gws, V, h->eps,
                                 h->rotcnt, h->info, s0));
    return 0;
}
}  // extern "C++"

extern "C++" {
template <int EPL, bool HALF = false>
static int launch_jacobi_smem_t(pfsm_ctx* h, const double* A, double* V, cudaStream_t st, int32_t s0, int32_t ns,
                                int32_t compact) {
    SliceTable tab{h->slice_tab, h->slice_tab + h->P, h->slice_tab + 2 * (size_t)h->P, h->slice_tab + 3 * (size_t)h->P};
    const size_t smem = jacobi_smem_bytes(h->M, h->jac_hloc);
    // static smem (~300 B) + dynamic must stay within the 227 KB opt-in limit; set per launch (handles differ)
    PFSM_CUDA(cudaFuncSetAttribute(jacobi_smem_kernel<EPL, HALF>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3((unsigned)(ns * h->jac_cs));
    cfg.blockDim = dim3(HALF ? 512 : jacobi_smem_threads(EPL));
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)h->jac_cs;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    PFSM_CUDA(cudaLaunchKernelEx(&cfg, jacobi_smem_kernel<EPL, HALF>, A, h->ld, h->M, (int32_t)h->jac_hloc, tab,
                                 h->nrm_g, V, h->eps, h->rotcnt, h->info, s0, compact));
    return 0;
}
}  // extern "C++"

extern "C++" {
// how many clusters of `cs` CTAs of the shared-memory Jacobi kernel the device can hold at once
template <int EPL, bool HALF = false>
static int jacobi_max_clusters_t(int cs, size_t smem) {
    if (cudaFuncSetAttribute(jacobi_smem_kernel<EPL, HALF>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3((unsigned)cs);
    cfg.blockDim = dim3(HALF ? 512 : jacobi_smem_threads(EPL));
    cfg.dynamicSmemBytes = smem;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)cs;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, jacobi_smem_kernel<EPL, HALF>, &cfg) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    return n;
}
}  // extern "C++"

static int jacobi_max_clusters(int M, int cs, size_t smem, bool half = false) {
    if (half) {
        switch (jacobi_padded_rows(M) / 32) {
            case 2: return jacobi_max_clusters_t<2, true>(cs, smem);
            case 4: return jacobi_max_clusters_t<4, true>(cs, smem);
            case 6: return jacobi_max_clusters_t<6, true>(cs, smem);
            case 8: return jacobi_max_clusters_t<8, true>(cs, smem);
            default: return 0;
        }
    }
    switch (jacobi_padded_rows(M) / 32) {
        case 2: return jacobi_max_clusters_t<2>(cs, smem);
        case 4: return jacobi_max_clusters_t<4>(cs, smem);
        case 6: return jacobi_max_clusters_t<6>(cs, smem);
        case 8: return jacobi_max_clusters_t<8>(cs, smem);
        case 10: return jacobi_max_clusters_t<10>(cs, smem);
        case 12: return jacobi_max_clusters_t<12>(cs, smem);
        case 14: return jacobi_max_clusters_t<14>(cs, smem);
        default: return jacobi_max_clusters_t<16>(cs, smem);
    }
}

// Shared-memory Jacobi layout.  The kernel is bound by the dependent chain of a round (load, reduce, rotate,
// exchange: ~1.2 us whatever the number of pairs a CTA holds), so more CTAs per slice help only while all P
// clusters are co-resident: the largest cluster size in {1,2,4,8} that fits the column slots in shared memory,
// leaves a CTA at least 6 pairs, and keeps the launch in ONE wave (cudaOccupancyMaxActiveClusters); if no size
// gives one wave, the smallest that fits.  0 = use the L2-resident kernel.
static void choose_jacobi_layout(pfsm_ctx* h) {
    h->jac_cs = 0;
    h->jac_hloc = 0;
    h->jac_half = false;
    h->jac_wide = h->opt_route == 3 && h->M <= JW_MAX_M;  // option step2_route = 3: the persistent-grid Jacobi kernel (M <= 4096)
    // Route of step 2.  Tridiagonalization + bisection + inverse iteration + back-transformation costs ~M latency-bound
    // columns; the Jacobi kernels cost sweeps x (M - 1) rounds.  With the submatrix resident in the cluster's distributed
    // shared memory (sytrd_dsmem_kernel) the tridiagonal route wins at every size measured (step 2, Jacobi -> tridiagonal):
    // M = 32 x 8 slices 0.20 -> 0.17 ms, 64 x 64 0.55 -> 0.34, 96 x 4 0.61 -> 0.46, 128 x 32 1.29 -> 0.68, 160 x 4 1.39 -> 0.77,
    // 192 x 16 2.66 -> 1.10, 224 x 24 4.57 -> 1.46, 256 x 64 12.5 -> 3.4, 416 x 13 15.2 -> 2.65 ms.  So: the tridiagonal route
    // from M = 16 on; the shared-memory Jacobi only for tiny submatrices.
    // Option step2_route = 1 / 2 forces one family (M > 512 has no shared-memory / L2 Jacobi: step2_route = 3).
    const bool want_jacobi = h->opt_route == 1 && h->M <= 512;
    h->tridiag = !h->jac_wide && !want_jacobi && (h->M >= 16 || h->opt_route == 2);
    if (h->M > 512 || h->jac_wide || h->tridiag) return;
    if (h->opt_jacobi_l2) return;  // option jacobi_l2: force the L2-resident kernel (the large-M fallback)
    const size_t budget = 220 * 1024;
    // seats per CTA; one more (phantom) pair when seat 0 and seat h_loc-1 would fall to the same warp, because the
    // two boundary seats of a CTA synchronise with each other inside a round (jacobi_smem.cuh)
    const int epl = jacobi_padded_rows(h->M) / 32;
    auto hloc_of = [&](int cs, bool half = false) {
        int hl = (h->M + 2 * cs - 1) / (2 * cs);
        const int nw = (half ? 512 : jacobi_smem_threads(epl)) / 32;  // warps per CTA
        if (hl > 1 && (hl - 1) % nw == 0) ++hl;
        return hl;
    };
    auto fits = [&](int cs, bool half = false) {
        return hloc_of(cs, half) >= 2 && jacobi_smem_bytes(h->M, hloc_of(cs, half)) <= budget;
    };
    int cs_min = 1;
    while (cs_min <= 8 && !fits(cs_min)) cs_min *= 2;
    if (cs_min > 8) return;
    int cs = cs_min;
    bool one_wave = false;
    for (int c = cs_min; c <= 8; c *= 2) {
        if (!fits(c) || (c > cs_min && hloc_of(c) < 6)) break;
        if (jacobi_max_clusters(h->M, c, jacobi_smem_bytes(h->M, hloc_of(c))) >= h->P) { cs = c; one_wave = true; }
    }
    // More than one wave of full CTAs: clusters of 8 half CTAs (512 threads, one pair per warp, two CTAs of different
    // slices per SM) hold as many slices per wave and overlap each other's barrier and exchange waits.
    bool half = false;
    if (!one_wave && epl <= 8 && fits(8, true) && hloc_of(8, true) >= 6 && hloc_of(8, true) <= 16) {
        const int full_per_wave = jacobi_max_clusters(h->M, cs, jacobi_smem_bytes(h->M, hloc_of(cs)));
        const int half_per_wave = jacobi_max_clusters(h->M, 8, jacobi_smem_bytes(h->M, hloc_of(8, true)), true);
        auto waves = [&](int per) { return per > 0 ? (h->P + per - 1) / per : 1 << 20; };
        if (waves(half_per_wave) <= waves(full_per_wave) && !h->opt_jacobi_full) {  // option jacobi_full_cta: full CTAs only
            half = true;
            cs = 8;
        }
    }
    if (h->opt_jacobi_cs) {  // option jacobi_cluster_size: override
        const int want = h->opt_jacobi_cs;
        if ((want == 1 || want == 2 || want == 4 || want == 8) && fits(want, half)) cs = want;
    }
    h->jac_half = half;
    h->jac_cs = cs;
    h->jac_hloc = hloc_of(cs, half);
}

// Wide windows (512 < M <= 4096): one persistent cooperative grid over all slices (jacobi_wide.cuh)
extern "C++" {
template <int EPT>
static int launch_jacobi_wide_t(pfsm_ctx* h, const double* A, double* V, cudaStream_t st, int32_t s0, int32_t ns) {
    SliceTable tab{h->slice_tab, h->slice_tab + h->P, h->slice_tab + 2 * (size_t)h->P, h->slice_tab + 3 * (size_t)h->P};
    const size_t smem = (size_t)ns * sizeof(int);
    int per_sm = 0, sms = 0;
    PFSM_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, jacobi_wide_kernel<EPT>, JW_THREADS, smem));
    PFSM_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, h->device));
    if (per_sm < 1) return PFSM_CUDA_ERROR_BASE + (int)cudaErrorLaunchOutOfResources;
    const int64_t units = (int64_t)ns * ((h->M + 1) / 2);
    const int64_t want = (units + JW_GPC - 1) / JW_GPC;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((int64_t)per_sm * sms, want));
    PFSM_CUDA(cudaMemsetAsync(h->jw_bar, 0, sizeof(unsigned int), st));
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(JW_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;  // all CTAs co-resident: the grid barrier cannot deadlock
    attr[0].val.cooperative = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    PFSM_CUDA(cudaLaunchKernelEx(&cfg, jacobi_wide_kernel<EPT>, A, h->ld, h->M, tab, h->Gws, h->nrm_g, V, h->eps,
                                 h->rotcnt, h->info, s0, ns, h->jw_bar));
    return 0;
}
}  // extern "C++"

// Does step 2 of `ns` slices take the blocked tridiagonalization?  (See launch_tridiag for the measurements behind the rule.)
static bool uses_blocked_sytrd(const pfsm_ctx* h, int32_t ns) {
    const int64_t M = h->M;
    if (!h->tridiag || (M % 2) != 0 || M < 4 || M > 4096) return false;  // (M even: 16-byte pitch of the tensor maps; M <= 8 x 512 rows per thread)
    if (h->opt_sytrd_storage == 3) return true;
    if (h->opt_sytrd_storage != 0) return false;
    int l2b = 0;
    if (cudaDeviceGetAttribute(&l2b, cudaDevAttrL2CacheSize, h->device) != cudaSuccess) return false;
    return (size_t)ns * M * M * sizeof(double) > (size_t)l2b + (size_t)l2b / 2;
}

// ---- Blocked tridiagonalization (sytrd_blocked.cuh): per panel of SB_NB columns one cooperative launch of
// sytrd_panel_kernel (C CTAs per slice, per-slice barriers) and one batched rank-2NB trailing update on the DMMA pipe.
static int ensure_blocked_ws(pfsm_ctx* h) {
    if (h->sbw.VW) return 0;
    const int64_t M = h->M, P = h->P;
    int rc;
#define TRYA(x) do { if ((rc = (x))) return rc; } while (0)
    const size_t pm = (size_t)P * M * sizeof(double);
    TRYA(dev_alloc(h, (void**)&h->sbw.VW, pm * 2 * SB_NB));
    TRYA(dev_alloc(h, (void**)&h->sbw.WV, pm * 2 * SB_NB));
    TRYA(dev_alloc(h, (void**)&h->sbw.ypart, (size_t)h->sms * M * sizeof(double)));
    TRYA(dev_alloc(h, (void**)&h->sbw.y, 2 * pm));
    TRYA(dev_alloc(h, (void**)&h->sbw.base, 2 * pm));
    TRYA(dev_alloc(h, (void**)&h->sbw.dots, (size_t)h->sms * 2 * SB_NB * sizeof(double)));
    TRYA(dev_alloc(h, (void**)&h->sbw.yv, (size_t)2 * h->sms * sizeof(double)));
    TRYA(dev_alloc(h, (void**)&h->sbw.sbar, (size_t)P * sizeof(unsigned int)));
    PFSM_CUDA(cudaMemset(h->sbw.VW, 0, pm * 2 * SB_NB));
    PFSM_CUDA(cudaMemset(h->sbw.WV, 0, pm * 2 * SB_NB));
    TRYA(make_map(&h->mapG, h->Gws, P * M, M, M));
    TRYA(make_map(&h->mapVW, h->sbw.VW, P * M, 2 * SB_NB, 2 * SB_NB));
    TRYA(make_map(&h->mapWV, h->sbw.WV, P * M, 2 * SB_NB, 2 * SB_NB));
#undef TRYA
    return 0;
}

static int launch_sytrd_blocked(pfsm_ctx* h, const double* A, cudaStream_t st, int32_t s0, int32_t ns, int32_t precopied) {
    SliceTable tab{h->slice_tab, h->slice_tab + h->P, h->slice_tab + 2 * (size_t)h->P, h->slice_tab + 3 * (size_t)h->P};
    const int M = h->M;
    int rc;
    if ((rc = ensure_blocked_ws(h))) return rc;
    if (!precopied) {
        sytrd_copy_kernel<<<dim3((unsigned)M, (unsigned)ns), 256, 0, st>>>(A, h->ld, M, tab, h->Gws, s0);
        PFSM_CUDA(cudaGetLastError());
    }
    const int nbk = (M + 31) / 32;
    const int cap = h->sms;  // one CTA per SM (shared memory)
    for (int sb0 = 0; sb0 < ns; sb0 += cap) {  // more slices than SMs: batches of slices, one CTA each
        const int nsl = std::min(ns - sb0, cap);
        const int C = std::max(1, std::min(cap / nsl, nbk));
        // shared-memory slots: one chunk per column if it fits, never less than one strip
        const size_t budget = 200 * 1024;
        int slot_tiles = std::max(sb_max_tiles_per_cta(M, C), nbk);
        while (slot_tiles > nbk && sb_smem_bytes(M, slot_tiles) > budget) --slot_tiles;
        const size_t smem = sb_smem_bytes(M, slot_tiles);
        PFSM_CUDA(cudaFuncSetAttribute(sytrd_panel_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        for (int k0 = 0; k0 < M - 1; k0 += SB_NB) {
            const int ncols = std::min(SB_NB, M - 1 - k0);
            PFSM_CUDA(cudaMemsetAsync(h->sbw.sbar + s0 + sb0, 0, (size_t)nsl * sizeof(unsigned int), st));
            cudaLaunchConfig_t cfg;
            memset(&cfg, 0, sizeof(cfg));
            cfg.gridDim = dim3((unsigned)(nsl * C));
            cfg.blockDim = dim3(SB_THREADS);
            cfg.dynamicSmemBytes = smem;
            cfg.stream = st;
            cudaLaunchAttribute attr[1];
            attr[0].id = cudaLaunchAttributeCooperative;  // all CTAs co-resident: the slice barriers cannot deadlock
            attr[0].val.cooperative = 1;
            cfg.attrs = attr;
            cfg.numAttrs = 1;
            PFSM_CUDA(cudaLaunchKernelEx(&cfg, sytrd_panel_kernel, h->Gws, (int32_t)M, h->tri, h->sbw, h->P,
                                         (int32_t)(s0 + sb0), (int32_t)C, (int32_t)k0, (int32_t)ncols, (int32_t)slot_tiles));
            const int kt = k0 + SB_NB;
            if (kt < M - 1) {  // A[kt:, kt:] -= V W^T + W V^T on the lower tiles, all slices of the batch in one launch
                GemmParams p = base_params();
                p.C = h->Gws; p.ldc = M; p.cr0 = (s0 + sb0) * M + kt; p.cc0 = kt; p.mr = M - kt; p.nc = M - kt;
                p.xr0 = (s0 + sb0) * M + kt; p.yr0 = (s0 + sb0) * M + kt; p.klen = 2 * SB_NB; p.lower = 1;
                p.nbatch = nsl; p.bxs = M; p.bys = M; p.bcs = M;
                if ((rc = launch_gemm<EPI_SUB>(h, h->mapVW, h->mapWV, h->mapG, p, st))) return rc;
            }
        }
    }
    return 0;
}

// Wide windows, default route: Householder tridiagonalization + bisection + inverse iteration + back-transformation
static int launch_tridiag(pfsm_ctx* h, const double* A, double* V, cudaStream_t st, int32_t s0, int32_t ns, int32_t precopied) {
    SliceTable tab{h->slice_tab, h->slice_tab + h->P, h->slice_tab + 2 * (size_t)h->P, h->slice_tab + 3 * (size_t)h->P};
    const int M = h->M;
    int sms = 0;
    PFSM_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, h->device));
    // Blocked route (panel + DMMA rank-2NB update; M even: the tensor maps need a 16-byte pitch).  Its read-only pass per
    // column halves the HBM traffic of the lower-triangle kernel but costs two slice barriers and more O(M) work per column,
    // so it wins once the batch is well beyond L2 (step 2, full / lower / blocked: 1536 x 8 = 151 MB 45 / 42 / 42 ms,
    // 2048 x 8 = 268 MB 96 / 80 / 69, 2048 x 16 = 537 MB 163 / 120 / 83; 2048 x 4 = 134 MB 60 / 61 / 75).
    const bool blocked = uses_blocked_sytrd(h, ns);
    if (blocked) {
        int rcb;
        if ((rcb = launch_sytrd_blocked(h, A, st, s0, ns, precopied))) return rcb;
    } else
    {
        const size_t smem = 3 * (size_t)M * sizeof(double);
        // Lower-triangle storage halves the HBM traffic but pays a second grid barrier and a partial-sum pass per
        // column: it wins once the batch of submatrices no longer fits L2 (M = 2048 x 16: 147 -> 104 ms; M = 1024 x 4,
        // L2 resident: 11 -> 17 ms, so full storage is kept there)
        int l2 = 0;
        PFSM_CUDA(cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, h->device));
        // (the full-storage kernel holds row k in 8 registers per thread: M <= 4096; beyond, the lower-triangle kernel)
        const bool half = M > 4096 || (h->opt_sytrd_storage != 1 && (h->opt_sytrd_storage == 2 || (size_t)ns * M * M * sizeof(double) > (size_t)l2));
        // Small submatrices (a column is latency bound): the CTAs of a slice form a cluster and use its barrier
        const bool small = !half && M <= 768 && h->opt_sytrd_grid != 1;
        bool cluster = small;
        int ccl = 1;  // cluster size: the largest of 8, 4, 2 that keeps all ns clusters co-resident (one wave)
        if (cluster) {
            PFSM_CUDA(cudaFuncSetAttribute(sytrd_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            cluster = false;
            for (int c2 = 8; c2 >= 2 && !cluster; c2 /= 2) {
                if (c2 * 16 > M + 15) continue;
                cudaLaunchConfig_t q;
                memset(&q, 0, sizeof(q));
                q.gridDim = dim3((unsigned)(ns * c2));
                q.blockDim = dim3(TRD_THREADS);
                q.dynamicSmemBytes = smem;
                cudaLaunchAttribute qa[1];
                qa[0].id = cudaLaunchAttributeClusterDimension;
                qa[0].val.clusterDim.x = (unsigned)c2;
                qa[0].val.clusterDim.y = 1;
                qa[0].val.clusterDim.z = 1;
                q.attrs = qa;
                q.numAttrs = 1;
                int nmax = 0;
                if (cudaOccupancyMaxActiveClusters(&nmax, sytrd_kernel<true>, &q) != cudaSuccess) { (void)cudaGetLastError(); break; }
                if (nmax >= ns) { cluster = true; ccl = c2; }
            }
        }
        // Small submatrices: resident in the distributed shared memory of the slice's cluster (sytrd_dsmem_kernel) when some
        // cluster size fits 8 M^2 / C bytes per CTA; the size with the fewest waves wins (a column is latency bound whatever
        // C is), ties go to the larger cluster.  Option sytrd_grid_barrier = 2 keeps the L2-resident cluster kernel.
        int dsC = 0;
        if (small && h->opt_sytrd_grid != 2) {
            int best_waves = INT_MAX;
            for (int c2 = 8; c2 >= 1; c2 /= 2) {
                if (c2 > 1 && c2 * 16 > M + 15) continue;
                const size_t sm = sytrd_dsmem_bytes(M, c2);
                if (sm > (size_t)220 * 1024) continue;
                if (cudaFuncSetAttribute(sytrd_dsmem_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm) != cudaSuccess) {
                    (void)cudaGetLastError();
                    continue;
                }
                cudaLaunchConfig_t q;
                memset(&q, 0, sizeof(q));
                q.gridDim = dim3((unsigned)(ns * c2));
                q.blockDim = dim3(TRD_THREADS);
                q.dynamicSmemBytes = sm;
                cudaLaunchAttribute qa[1];
                qa[0].id = cudaLaunchAttributeClusterDimension;
                qa[0].val.clusterDim.x = (unsigned)c2;
                qa[0].val.clusterDim.y = 1;
                qa[0].val.clusterDim.z = 1;
                q.attrs = qa;
                q.numAttrs = 1;
                int nmax = 0;
                if (cudaOccupancyMaxActiveClusters(&nmax, sytrd_dsmem_kernel, &q) != cudaSuccess || nmax < 1) { (void)cudaGetLastError(); continue; }
                const int waves = (ns + nmax - 1) / nmax;
                if (waves < best_waves) { best_waves = waves; dsC = c2; }
            }
            // measured (step 2, DSMEM / L2-resident): 16 x 192 1.10 / 1.50 ms, 24 x 224 1.46 / 1.99, 13 x 416 2.65 / 3.93,
            // 64 x 256 (2 waves) 3.43 / 3.54, 72 x 254 (3 waves) 4.52 / 4.33: beyond two waves the L2-resident kernel, whose
            // clusters are all co-resident, is the faster one
            if (best_waves > 2) dsC = 0;
        }
        if (dsC > 0) {
            const size_t sm = sytrd_dsmem_bytes(M, dsC);
            PFSM_CUDA(cudaFuncSetAttribute(sytrd_dsmem_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
            cudaLaunchConfig_t cfg;
            memset(&cfg, 0, sizeof(cfg));
            cfg.gridDim = dim3((unsigned)(ns * dsC));
            cfg.blockDim = dim3(TRD_THREADS);
            cfg.dynamicSmemBytes = sm;
            cfg.stream = st;
            cudaLaunchAttribute attr[1];
            attr[0].id = cudaLaunchAttributeClusterDimension;
            attr[0].val.clusterDim.x = (unsigned)dsC;
            attr[0].val.clusterDim.y = 1;
            attr[0].val.clusterDim.z = 1;
            cfg.attrs = attr;
            cfg.numAttrs = 1;
            PFSM_CUDA(cudaLaunchKernelEx(&cfg, sytrd_dsmem_kernel, A, h->ld, (int32_t)M, tab, h->Gws, h->tri, h->P, s0, (int32_t)dsC, precopied));
        } else {
        auto kern = half ? sytrd_half_kernel : (cluster ? sytrd_kernel<true> : sytrd_kernel<false>);
        PFSM_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int per_sm = 0;
        PFSM_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, TRD_THREADS, smem));
        if (per_sm < 1) return PFSM_CUDA_ERROR_BASE + (int)cudaErrorLaunchOutOfResources;
        const int cap = per_sm * sms;
        int C = std::max(1, std::min(cap / ns, (M + 15) / 16));  // CTAs per slice; a CTA keeps >= 16 rows while rows last
        if (cluster) C = ccl;
        const int grid = cluster ? ns * C : std::min(cap, ns * C);
        cudaLaunchConfig_t cfg;
        memset(&cfg, 0, sizeof(cfg));
        cfg.gridDim = dim3((unsigned)grid);
        cfg.blockDim = dim3(TRD_THREADS);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        if (cluster) {
            attr[0].id = cudaLaunchAttributeClusterDimension;
            attr[0].val.clusterDim.x = (unsigned)C;
            attr[0].val.clusterDim.y = 1;
            attr[0].val.clusterDim.z = 1;
        } else {
            PFSM_CUDA(cudaMemsetAsync(h->jw_bar, 0, sizeof(unsigned int), st));
            attr[0].id = cudaLaunchAttributeCooperative;  // all CTAs co-resident: the grid barrier cannot deadlock
            attr[0].val.cooperative = 1;
        }
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        PFSM_CUDA(cudaLaunchKernelEx(&cfg, kern, A, h->ld, (int32_t)M, tab, h->Gws, h->tri, h->P, s0, ns, (int32_t)C,
                                     h->jw_bar, precopied));
    }
        }
    const size_t smem2 = 2 * (size_t)M * sizeof(double);
    PFSM_CUDA(cudaFuncSetAttribute(tri_bisect_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2));
    PFSM_CUDA(cudaFuncSetAttribute(tri_invit_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2));
    const dim3 g2((unsigned)((h->m + TRI_THREADS - 1) / TRI_THREADS), (unsigned)ns);
    const dim3 g2b((unsigned)((h->m + TRI_THREADS / 32 - 1) / (TRI_THREADS / 32)), (unsigned)ns);
    tri_bisect_kernel<<<g2b, TRI_THREADS, smem2, st>>>((int32_t)M, tab, h->tri, s0);
    PFSM_CUDA(cudaGetLastError());
    tri_invit_kernel<<<g2, TRI_THREADS, smem2, st>>>(h->ld, (int32_t)M, tab, h->tri, s0, h->info);
    PFSM_CUDA(cudaGetLastError());
    {   // re-orthogonalization inside tight eigenvalue clusters: the runs of a slice are dealt to CX CTAs
        const bool staged = M <= TRC_STAGED_MAX_M;
        const size_t smem3 = tri_cluster_smem_bytes(M, h->m, staged);
        const int cx = std::max(1, std::min(64, (2 * h->sms) / std::max(1, ns)));
        const dim3 g4((unsigned)cx, (unsigned)ns);
        if (staged) {
            PFSM_CUDA(cudaFuncSetAttribute(tri_cluster_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem3));
            tri_cluster_kernel<true><<<g4, TRC_THREADS, smem3, st>>>(h->ld, (int32_t)M, tab, h->tri, s0, h->m);
        } else {
            PFSM_CUDA(cudaFuncSetAttribute(tri_cluster_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem3));
            tri_cluster_kernel<false><<<g4, TRC_THREADS, smem3, st>>>(h->ld, (int32_t)M, tab, h->tri, s0, h->m);
        }
        PFSM_CUDA(cudaGetLastError());
    }
    {
        const int ept = (M + BT_THREADS - 1) / BT_THREADS;
        const int nvec = ept <= 8 ? 8 : (ept <= 16 ? 4 : 2);
        const dim3 g3((unsigned)((h->m + nvec - 1) / nvec), (unsigned)ns);
#define PFSM_BT(E, NVEC) tri_backtransform_kernel<E, NVEC><<<g3, BT_THREADS, 0, st>>>(h->ld, (int32_t)M, tab, h->Gws, h->tri, V, h->eps, s0)
        if (ept <= 1) PFSM_BT(1, 8);
        else if (ept <= 2) PFSM_BT(2, 8);
        else if (ept <= 4) PFSM_BT(4, 8);
        else if (ept <= 6) PFSM_BT(6, 8);
        else if (ept <= 8) PFSM_BT(8, 8);
        else if (ept <= 12) PFSM_BT(12, 4);
        else if (ept <= 16) PFSM_BT(16, 4);
        else if (ept <= 24) PFSM_BT(24, 2);
        else PFSM_BT(32, 2);
#undef PFSM_BT
        PFSM_CUDA(cudaGetLastError());
    }
    return 0;
}

static int launch_jacobi(pfsm_ctx* h, const double* A, double* V, cudaStream_t st, int32_t s0 = 0, int32_t ns = -1,
                         int32_t compact = 0) {
    if (ns < 0) ns = h->P;
    PFSM_CUDA(cudaMemsetAsync(h->rotcnt, 0, (size_t)h->P * JACOBI_MAX_SWEEPS * sizeof(int), st));
    if (h->tridiag) return launch_tridiag(h, A, V, st, s0, ns, compact);
    if (h->M > 512 || h->jac_wide) {
        const int ept = (h->M + JW_GROUP - 1) / JW_GROUP;
        if (ept <= 2) return launch_jacobi_wide_t<2>(h, A, V, st, s0, ns);
        if (ept <= 4) return launch_jacobi_wide_t<4>(h, A, V, st, s0, ns);
        if (ept <= 6) return launch_jacobi_wide_t<6>(h, A, V, st, s0, ns);
        if (ept <= 8) return launch_jacobi_wide_t<8>(h, A, V, st, s0, ns);
        if (ept <= 12) return launch_jacobi_wide_t<12>(h, A, V, st, s0, ns);
        return launch_jacobi_wide_t<16>(h, A, V, st, s0, ns);
    }
    if (h->jac_cs > 0 && h->jac_half) {
        switch (jacobi_padded_rows(h->M) / 32) {
            case 2: return launch_jacobi_smem_t<2, true>(h, A, V, st, s0, ns, compact);
            case 4: return launch_jacobi_smem_t<4, true>(h, A, V, st, s0, ns, compact);
            case 6: return launch_jacobi_smem_t<6, true>(h, A, V, st, s0, ns, compact);
            default: return launch_jacobi_smem_t<8, true>(h, A, V, st, s0, ns, compact);
        }
    }
    if (h->jac_cs > 0) {
        switch (jacobi_padded_rows(h->M) / 32) {  // doubles per lane per column
            case 2: return launch_jacobi_smem_t<2>(h, A, V, st, s0, ns, compact);
            case 4: return launch_jacobi_smem_t<4>(h, A, V, st, s0, ns, compact);
            case 6: return launch_jacobi_smem_t<6>(h, A, V, st, s0, ns, compact);
            case 8: return launch_jacobi_smem_t<8>(h, A, V, st, s0, ns, compact);
            case 10: return launch_jacobi_smem_t<10>(h, A, V, st, s0, ns, compact);
            case 12: return launch_jacobi_smem_t<12>(h, A, V, st, s0, ns, compact);
            case 14: return launch_jacobi_smem_t<14>(h, A, V, st, s0, ns, compact);
            default: return launch_jacobi_smem_t<16>(h, A, V, st, s0, ns, compact);
        }
    }
    if (h->M <= 128) return launch_jacobi_t<4>(h, A, V, st, s0, ns);
    if (h->M <= 256) return launch_jacobi_t<8>(h, A, V, st, s0, ns);
    return launch_jacobi_t<16>(h, A, V, st, s0, ns);
}

// Groups of panels of the stacked Cholesky (see stacked_cholesky): boundaries in panel units, last entry = nblk.
static std::vector<int32_t> chol_group_bounds(const pfsm_ctx* h) {
    std::vector<int32_t> gb;
    const int32_t big = h->opt_chol_group ? h->opt_chol_group : (h->nblk >= 48 ? 4 : 2);
    const int32_t tail = 24;  // panels at the end that stay in pairs (measured flat between 16 and 24 at N = 8192)
    for (int32_t k = 0; k < h->nblk;) {
        gb.push_back(k);
        k += (big > 2 && h->nblk - k > tail) ? big : 2;
    }
    gb.push_back(h->nblk);
    return gb;
}

// ---- Stacked right-looking Cholesky on S = [G ; Z] (2N x N, row-major view): O = [L ; Z L^-T] with G = L L^T.
// The panel step O[r,k] = S[r,k] L_kk^-T and the trailing update S[r,c] -= O[r,k] O[c,k]^T run over every row
// below the diagonal block, so the triangular solve of the bottom rows is folded into the factorization's GEMMs.
// factor = false re-uses L (O's top) and the inverted diagonal blocks of an earlier pass and only transforms
// the bottom rows [N, 2N).  Two-level blocking: 128-wide panels are factored one by one, but the big trailing
// update is applied once per PAIR of panels with K = 256, halving how often every C tile is read and re-written.
// b0, b1: only the bottom rows [N + b0, N + b1) are transformed (a rank of the sharded solve owns a row block of Z).
// peer_bottom: the transformed bottom rows are also stored into the other ranks' copies of O (peer-write mode).
static int stacked_cholesky(pfsm_ctx* h, bool factor, cudaStream_t st, int32_t b0 = 0, int32_t b1 = -1, bool peer_bottom = false) {
    const int64_t N = h->N, L = h->ld;
    const int32_t n = (int32_t)N;
    if (b1 < 0) b1 = n;
    const bool whole = factor && b0 == 0 && b1 == n;  // top and bottom rows form one contiguous row range
    int rc;
    if (!h->chol_attr) {
        PFSM_CUDA(cudaFuncSetAttribute(chol_diag_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, CHOL_SMEM));
        h->chol_attr = true;
    }
    cudaStream_t cs = st;  // stream the helpers below launch on (switched by the look-ahead schedule)
    // panel rows [r0, r0 + nr): O[r, k0:k0+nb] = S[r, k0:k0+nb] L_kk^-T
    auto panel_rows = [&](int32_t k, int32_t r0, int32_t nr) -> int {
        if (nr <= 0) return 0;
        const int32_t k0 = k * CHOL_NB, nb = (int32_t)std::min<int64_t>(CHOL_NB, N - k0);
        GemmParams pp = base_params();
        pp.C = h->O; pp.ldc = L; pp.cr0 = r0; pp.cc0 = k0; pp.mr = nr; pp.nc = nb;
        pp.xr0 = r0; pp.xk0 = k0; pp.yr0 = k * CHOL_NB; pp.yk0 = 0; pp.klen = nb;
        if (peer_bottom && h->npeer > 0 && r0 >= n) {  // (peer_buf[2] points at the peer's row N of O: same coordinates as h->O)
            pp.npeer = h->npeer;
            for (int i = 0; i < h->npeer; ++i) pp.peerC[i] = h->peer_buf[2][i] - (size_t)N * L;
            return launch_gemm<EPI_PLAIN, true>(h, h->mapS, h->mapD, h->mapO, pp, cs);
        }
        return launch_gemm<EPI_PLAIN>(h, h->mapS, h->mapD, h->mapO, pp, cs);
    };
    auto factor_panel = [&](int32_t k) -> int {
        const int32_t k0 = k * CHOL_NB, nb = (int32_t)std::min<int64_t>(CHOL_NB, N - k0);
        if (factor) {
            chol_diag_kernel<<<1, CHOL_THREADS, CHOL_SMEM, cs>>>(h->S, h->O, L, k0, nb,
                                                                 h->Dinv + (size_t)k * CHOL_NB * CHOL_NB, h->gdiag, h->info);
            PFSM_CUDA(cudaGetLastError());
        }
        if (whole) return panel_rows(k, k0 + nb, 2 * n - k0 - nb);
        int r = factor ? panel_rows(k, k0 + nb, n - k0 - nb) : 0;   // rows of G below the diagonal block
        return r ? r : panel_rows(k, n + b0, b1 - b0);              // this call's rows of the bottom part
    };
    // rows [r0, r0 + nr): S[r, c0:c0+ncols] -= O[r, kk0:kk0+klen] . O[c, kk0:kk0+klen]
    auto update_rows = [&](int32_t r0, int32_t nr, int32_t c0, int32_t ncols, int32_t kk0, int32_t klen, int lower) -> int {
        if (ncols <= 0 || nr <= 0) return 0;
        GemmParams pt = base_params();
        pt.C = h->S; pt.ldc = L; pt.cr0 = r0; pt.cc0 = c0; pt.mr = nr; pt.nc = ncols;
        pt.xr0 = r0; pt.yr0 = c0; pt.xk0 = kk0; pt.yk0 = kk0; pt.klen = klen; pt.lower = lower;
        return launch_gemm<EPI_SUB>(h, h->mapO, h->mapO, h->mapS, pt, cs);
    };
    // columns [c0, c0 + ncols) of every active row at or below row c0 (lower tiles only where the region is square)
    auto update = [&](int32_t c0, int32_t ncols, int32_t kk0, int32_t klen, int lower) -> int {
        if (whole) return update_rows(c0, 2 * n - c0, c0, ncols, kk0, klen, lower);
        int r = factor ? update_rows(c0, n - c0, c0, ncols, kk0, klen, lower) : 0;
        return r ? r : update_rows(n + b0, b1 - b0, c0, ncols, kk0, klen, 0);
    };
    // Panels are factored one by one, but the big trailing update is applied once per GROUP of panels (K = 128 x group
    // size), which divides how often every C tile is read and re-written: groups of opt_chol_group panels (4: K = 512)
    // while many panels remain, pairs near the end, where the serial chain of a group is no longer hidden by its bulk update.
    const std::vector<int32_t> gb = chol_group_bounds(h);  // first panel of each group; last entry = nblk
    const int32_t npairs = (int32_t)gb.size() - 1;         // number of groups
    auto pair_c0 = [&](int32_t p) {                        // first column of group p
        return std::min<int32_t>(n, gb[std::min<size_t>((size_t)p, gb.size() - 1)] * CHOL_NB);
    };
    // the serial chain of group p: for each of its panels, bring the panel's columns up to date with the group's earlier
    // panels (left-looking inside the group, K = 128 .. 384), then factor it
    auto chain = [&](int32_t p) -> int {
        const int32_t kb = gb[p], ke = gb[p + 1];
        for (int32_t k = kb; k < ke; ++k) {
            int r;
            if (k > kb) {
                const int32_t k1 = k * CHOL_NB, nb1 = (int32_t)std::min<int64_t>(CHOL_NB, N - k1);
                if ((r = update(k1, nb1, kb * CHOL_NB, (k - kb) * CHOL_NB, 0))) return r;
            }
            if ((r = factor_panel(k))) return r;
        }
        return 0;
    };
    // columns [c0, c1) of the trailing matrix updated with group p's panels
    auto trailing = [&](int32_t p, int32_t c0, int32_t c1) -> int {
        const int32_t k0 = pair_c0(p), kend = pair_c0(p + 1);
        return update(c0, c1 - c0, k0, kend - k0, 1);
    };
    if (whole && h->lookahead && npairs >= 3) {
        // Look-ahead: while the main stream applies pair p's update to the bulk of the trailing matrix, a
        // high-priority side stream updates just the next pair's 256 columns and runs that pair's serial chain
        // (diagonal-block kernels and under-filled panel GEMMs), so the chain hides behind the bulk update.
        PFSM_CUDA(cudaEventRecord(h->ev_fork, st));
        PFSM_CUDA(cudaStreamWaitEvent(h->side, h->ev_fork, 0));
        cs = h->side;
        if ((rc = chain(0))) return rc;
        PFSM_CUDA(cudaEventRecord(h->ev_chain, h->side));
        for (int32_t p = 0; p < npairs; ++p) {
            const int32_t cn0 = pair_c0(p + 1), cn1 = pair_c0(p + 2);
            PFSM_CUDA(cudaStreamWaitEvent(st, h->ev_chain, 0));      // main needs pair p's panels
            if (cn0 < n) {
                cs = h->side;                                        // side: next pair's columns, then its chain
                if (p > 0) PFSM_CUDA(cudaStreamWaitEvent(h->side, h->ev_rest, 0));  // ... on top of update p-1
                if ((rc = trailing(p, cn0, cn1))) return rc;
                if ((rc = chain(p + 1))) return rc;
                PFSM_CUDA(cudaEventRecord(h->ev_chain, h->side));
            }
            if (cn1 < n) {
                cs = st;                                             // main: the bulk of pair p's update
                if ((rc = trailing(p, cn1, n))) return rc;
                PFSM_CUDA(cudaEventRecord(h->ev_rest, st));
            }
        }
        PFSM_CUDA(cudaStreamWaitEvent(st, h->ev_chain, 0));          // join
        return 0;
    }
    for (int32_t p = 0; p < npairs; ++p) {
        if ((rc = chain(p))) return rc;
        const int32_t cn0 = pair_c0(p + 1);
        if (cn0 < n && (rc = trailing(p, cn0, n))) return rc;
    }
    return 0;
}

// ---- step 4: Cholesky-QR.  G = V^T V (row-major view: V V^T), S = [G ; V^T] ----
// wait_cnt != nullptr: V is the output of a step-3 GEMM that may still be in its last wave; the Gram product is chained
// to it (row-block counters, see the step-3 loop) and starts on the SMs that wave leaves idle.
static int run_step4_once(pfsm_ctx* h, const CUtensorMap& mapV, double* V, cudaStream_t st,
                          const int32_t* wait_cnt = nullptr, int32_t wait_target = 0) {
    const int64_t N = h->N, L = h->ld;
    const int32_t n = (int32_t)N;
    int rc;
    const dim3 tb(32, 8), tg((unsigned)((N + 31) / 32), (unsigned)((N + 31) / 32));
    GemmParams p = base_params();
    p.C = h->S; p.ldc = L; p.mr = n; p.nc = n; p.klen = n; p.lower = 2;
    p.wait_cnt = wait_cnt; p.wait_target = wait_target;
    if (wait_cnt) {
        if ((rc = launch_gemm<EPI_PLAIN>(h, mapV, mapV, h->mapS, p, st, true))) return rc;
    }
    transpose_kernel<<<tg, tb, 0, st>>>(V, L, h->S + (size_t)N * L, L, n, n);
    PFSM_CUDA(cudaGetLastError());
    if (!wait_cnt) {
        if ((rc = launch_gemm<EPI_PLAIN>(h, mapV, mapV, h->mapS, p, st))) return rc;
    }
    extract_diag_kernel<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(h->S, L, n, h->gdiag);
    PFSM_CUDA(cudaGetLastError());
    if ((rc = stacked_cholesky(h, true, st))) return rc;
    transpose_kernel<<<tg, tb, 0, st>>>(h->O + (size_t)N * L, L, V, L, n, n);
    PFSM_CUDA(cudaGetLastError());
    return 0;
}

// One pass leaves ||V^T V - I|| ~ eps cond(V)^2; a second pass on the result (CholeskyQR2) brings it to ~eps and does
// not change the exact-arithmetic result (V R1^-1 R2^-1 with R2 -> I), so it stays the Gram-Schmidt basis.
static int run_step4(pfsm_ctx* h, const CUtensorMap& mapV, double* V, cudaStream_t st,
                     const int32_t* wait_cnt = nullptr, int32_t wait_target = 0) {
    for (int32_t pass = 0; pass < h->cholqr_passes; ++pass) {
        int rc = pass == 0 ? run_step4_once(h, mapV, V, st, wait_cnt, wait_target) : run_step4_once(h, mapV, V, st);
        if (rc) return rc;
    }
    return 0;
}

// The kernel reads rows v_i and t_i twice (lambda_i first, then the residual).  With 8 blocks per SM the rows in flight
// (148 x 8 x 16 N bytes = 155 MB at N = 8192) outgrow the 126 MB L2 and the second read goes to HBM (ncu: 2.0 GB read for
// 1.07 GB of operands); a dynamic shared-memory reservation caps residency at 3 blocks per SM so the rows stay in L2.
static int launch_rayleigh(pfsm_ctx* h, const double* V, double* lambda_out, int32_t r0, int32_t rows, cudaStream_t st) {
    static const size_t RAY_CAP_SMEM = 72 * 1024;
    const size_t in_flight = (size_t)h->sms * 8 * 16 * (size_t)h->N;
    const size_t smem = in_flight > ((size_t)48 << 20) ? RAY_CAP_SMEM : 0;
    if (smem) PFSM_CUDA(cudaFuncSetAttribute(rayleigh_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    rayleigh_kernel<<<(unsigned)rows, RAY_THREADS, smem, st>>>(V, h->W, h->ld, h->N, lambda_out, h->resid, r0);
    PFSM_CUDA(cudaGetLastError());
    return 0;
}

// ---- step 5 (reading R11): T = V A, Rayleigh quotients and residual norms ----
static int run_step5(pfsm_ctx* h, const CUtensorMap& mapV, const CUtensorMap& mapA, double* V, double* lambda_out,
                     cudaStream_t st) {
    const int64_t N = h->N, L = h->ld;
    const int32_t n = (int32_t)N;
    int rc;
    {
        GemmParams p = base_params();
        p.C = h->W; p.ldc = L; p.mr = n; p.nc = n; p.klen = n;
        if ((rc = launch_gemm<EPI_PLAIN>(h, mapV, mapA, h->mapW, p, st))) return rc;
        if ((rc = launch_rayleigh(h, V, lambda_out, 0, n, st))) return rc;
    }
    return 0;
}

// ---- step 3 (Eq. 11) on rows [r0, r0 + rows) of the row-major V (eigenvectors r0 ..): two products per
// iteration.  Each product needs whole rows of the previous one's output, so the GEMMs are serial -- but only row block by
// row block: with 4096 tiles on 148 SMs the last wave of each is 100 tiles, and the next GEMM's first tiles (whose row
// blocks were finished waves ago) fill the idle SMs.  Hazards: tile (i, j) of GEMM g+1 overwrites what only tiles (i, .)
// of GEMM g read, and it starts after all of those have signalled.  A rank of the sharded solve runs the same chain on
// its own row range (rows / BM row blocks).  *last_cnt = the counters of the last update (nullptr when not chained).
// peers: the last update also stores its rows of V into the other ranks' V (peer-write mode of the sharded solve).
static int run_step3(pfsm_ctx* h, const CUtensorMap& mapV, const CUtensorMap& mapA, double* V, int32_t r0, int32_t rows,
                     cudaStream_t st, const int32_t** last_cnt, bool peers = false) {
    const int64_t N = h->N, L = h->ld;
    const int32_t n = (int32_t)N;
    const int32_t nrb = (rows + BM - 1) / BM, ncb = (n + BN - 1) / BN;
    const bool chain = h->chain && h->iters > 0;
    int rc;
    if (last_cnt) *last_cnt = nullptr;
    if (chain) PFSM_CUDA(cudaMemsetAsync(h->chain_cnt, 0, (size_t)2 * h->iters * nrb * sizeof(int32_t), st));
    for (int it = 0; it < h->iters; ++it) {
        GemmParams p = base_params();  // W = V A - diag(eps) V   (row-major view; A symmetric)
        p.C = h->W; p.ldc = L; p.cr0 = r0; p.xr0 = r0; p.mr = rows; p.nc = n; p.klen = n;
        p.krange = (it == 0) ? h->krange + r0 / BM : nullptr;  // start vectors are zero outside their window
        p.E1 = V; p.ld1 = L; p.eps = h->eps;
        GemmParams q = base_params();  // V <- V - alpha (W A - diag(eps) W)
        q.C = V; q.ldc = L; q.cr0 = r0; q.xr0 = r0; q.mr = rows; q.nc = n; q.klen = n;
        q.E1 = h->W; q.ld1 = L; q.E2 = V; q.ld2 = L; q.eps = h->eps; q.alpha = h->alpha;
        if (chain) {
            int32_t* c0 = h->chain_cnt + (size_t)(2 * it) * nrb;
            p.signal_cnt = c0;
            q.signal_cnt = c0 + nrb;
            q.wait_cnt = c0; q.wait_target = ncb;
            if (it > 0) { p.wait_cnt = c0 - nrb; p.wait_target = ncb; }
        }
        if ((rc = launch_gemm<EPI_SHIFT>(h, mapV, mapA, h->mapW, p, st, chain && it > 0))) return rc;
        if (peers && h->npeer > 0 && it == h->iters - 1) {
            q.npeer = h->npeer;
            for (int i = 0; i < h->npeer; ++i) q.peerC[i] = h->peer_buf[0][i];
            if ((rc = launch_gemm<EPI_UPDATE, true>(h, h->mapW, mapA, mapV, q, st, chain))) return rc;
        } else if ((rc = launch_gemm<EPI_UPDATE>(h, h->mapW, mapA, mapV, q, st, chain))) return rc;
    }
    if (chain && last_cnt) *last_cnt = h->chain_cnt + (size_t)(2 * h->iters - 1) * nrb;
    return 0;
}

// band != nullptr: packed copy of the P diagonal blocks for step 2 (A itself may still be in flight on the side
// stream; `a_ready` is waited for before step 3 reads it)
// A, V: leading dimension h->ld (the caller's own matrices when N is even, staged copies when it is odd)
static int solve_core(pfsm_handle_t h, const double* A, double* V, double* lambda_out, void* stream, int32_t last_step,
                      const double* band, cudaEvent_t a_ready) {
    if (!h) return -1;
    if (int rc_dev = check_device(h)) return rc_dev;
    if (!A || ((uintptr_t)A & 15)) return -2;
    if (!V || ((uintptr_t)V & 15)) return -3;
    if (last_step < 2 || last_step > 5) return -6;
    if (last_step == 5 && (!lambda_out || ((uintptr_t)lambda_out & 7))) return -4;
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t N = h->N, L = h->ld;
    const int32_t n = (int32_t)N;
    int rc;
    CUtensorMap mapA, mapV;
    if ((rc = make_map(&mapA, A, N, N, L))) return rc;
    if ((rc = make_map(&mapV, V, N, N, L))) return rc;
    const bool tm = h->timing;
    h->ev_valid = false;

    // ---- step 2: batched submatrix eigensolves -> shifts and zero-padded start vectors ----
    if (tm) PFSM_CUDA(cudaEventRecord(h->ev[0], st));
    if (!h->keep_info) PFSM_CUDA(cudaMemsetAsync(h->info, 0xFF, sizeof(unsigned long long), st));
    PFSM_CUDA(cudaMemsetAsync(V, 0, (size_t)N * L * sizeof(double), st));
    if ((rc = launch_jacobi(h, band ? band : A, V, st, 0, -1, band ? 1 : 0))) return rc;
    if (band) PFSM_CUDA(cudaStreamWaitEvent(st, a_ready, 0));
    if (tm) PFSM_CUDA(cudaEventRecord(h->ev[1], st));
    if (last_step == 2) return 0;

    // ---- step 3: folded-spectrum iterations (Eq. 11), two products per iteration ----
    const int32_t ncb = (n + BN - 1) / BN;
    const int32_t* step3_cnt = nullptr;
    if ((rc = run_step3(h, mapV, mapA, V, 0, n, st, &step3_cnt))) return rc;
    if (tm) PFSM_CUDA(cudaEventRecord(h->ev[2], st));
    if (last_step == 3) return 0;

    // The Gram product of step 4 is one more link of the chain: it reads row blocks of the last update.  Not with step
    // timing on: the event between the two kernels would sit inside the overlap and blur both step times.
    const int32_t* last_cnt = tm ? nullptr : step3_cnt;
    if ((rc = run_step4(h, mapV, V, st, last_cnt, ncb))) return rc;
    if (tm) PFSM_CUDA(cudaEventRecord(h->ev[3], st));
    if (last_step == 4) return 0;

    if ((rc = run_step5(h, mapV, mapA, V, lambda_out, st))) return rc;
    if (tm) {
        PFSM_CUDA(cudaEventRecord(h->ev[4], st));
        h->ev_valid = true;
    }
    return 0;
}

int pfsm_solve_partial(pfsm_handle_t h, const double* A, double* V, double* lambda_out, void* stream,
                       int32_t last_step) {
    if (!h) return -1;
    if (h->ld == h->N) return solve_core(h, A, V, lambda_out, stream, last_step, nullptr, nullptr);
    if (int rc_dev = check_device(h)) return rc_dev;
    if (!A || ((uintptr_t)A & 7)) return -2;
    if (!V || ((uintptr_t)V & 7)) return -3;
    cudaStream_t st = (cudaStream_t)stream;
    double *Au, *Vu;
    int rc;
    if ((rc = stage_in(h, A, &h->padA, &Au, st))) return rc;
    if ((rc = stage_in(h, V, &h->padV, &Vu, st, false))) return rc;
    if ((rc = solve_core(h, Au, Vu, lambda_out, stream, last_step, nullptr, nullptr))) return rc;
    return stage_out(h, Vu, V, st);
}

int pfsm_orthonormalize(pfsm_handle_t h, double* V_inout, void* stream) {
    if (!h) return -1;
    if (int rc_dev = check_device(h)) return rc_dev;
    if (!V_inout || ((uintptr_t)V_inout & (h->ld == h->N ? 15 : 7))) return -2;
    CUtensorMap mapV;
    int rc;
    cudaStream_t st = (cudaStream_t)stream;
    double* Vu;
    if ((rc = stage_in(h, V_inout, &h->padV, &Vu, st))) return rc;
    if ((rc = make_map(&mapV, Vu, h->N, h->N, h->ld))) return rc;
    h->ev_valid = false;
    PFSM_CUDA(cudaMemsetAsync(h->info, 0xFF, sizeof(unsigned long long), st));
    if ((rc = run_step4(h, mapV, Vu, st))) return rc;
    return stage_out(h, Vu, V_inout, st);
}

int pfsm_rayleigh(pfsm_handle_t h, const double* A, const double* V, double* lambda_out, void* stream) {
    if (!h) return -1;
    if (int rc_dev = check_device(h)) return rc_dev;
    const uintptr_t am = (h->ld == h->N) ? 15 : 7;
    if (!A || ((uintptr_t)A & am)) return -2;
    if (!V || ((uintptr_t)V & am)) return -3;
    if (!lambda_out || ((uintptr_t)lambda_out & 7)) return -4;
    CUtensorMap mapA, mapV;
    int rc;
    cudaStream_t st = (cudaStream_t)stream;
    double *Au, *Vu;
    if ((rc = stage_in(h, A, &h->padA, &Au, st))) return rc;
    if ((rc = stage_in(h, V, &h->padV, &Vu, st))) return rc;
    if ((rc = make_map(&mapA, Au, h->N, h->N, h->ld))) return rc;
    if ((rc = make_map(&mapV, Vu, h->N, h->N, h->ld))) return rc;
    h->ev_valid = false;
    return run_step5(h, mapV, mapA, Vu, lambda_out, st);
}

// ---- Row G (BASELINE.json configs[4], Eq. 13): A x = lambda S x reduced by Cholesky(S) ----
static int ensure_generalized(pfsm_ctx* h) {
    if (h->Ap) return 0;
    const int64_t N = h->N, L = h->ld;
    const size_t n2 = (size_t)N * L * sizeof(double);
    int rc;
    if ((rc = dev_alloc(h, (void**)&h->Ap, n2))) return rc;
    if ((rc = dev_alloc(h, (void**)&h->LT, n2))) return rc;
    if ((rc = dev_alloc(h, (void**)&h->DinvT, (size_t)h->nblk * CHOL_NB * CHOL_NB * sizeof(double)))) return rc;
    if ((rc = make_map(&h->mapAp, h->Ap, N, N, L))) return rc;
    if ((rc = make_map(&h->mapLT, h->LT, N, N, L))) return rc;
    if ((rc = make_map(&h->mapDT, h->DinvT, (int64_t)h->nblk * CHOL_NB, CHOL_NB, CHOL_NB))) return rc;
    return 0;
}

// S = L L^T;  Ap = L^-1 A L^-T (symmetrized);  keeps L^T and the transposed inverted diagonal blocks for the
// back-transformation.  Two passes of the stacked Cholesky: [S ; A] -> A L^-T, then [.; (A L^-T)^T] -> L^-1 A L^-T.
// A, S_in: the caller's matrices (leading dimension N); Ap_out: leading dimension ldo
static int run_generalized_reduce(pfsm_ctx* h, const double* A, const double* S_in, double* Ap_out, int64_t ldo, cudaStream_t st) {
    const int64_t N = h->N, L = h->ld;
    const int32_t n = (int32_t)N;
    int rc;
    const dim3 tb(32, 8), tg((unsigned)((N + 31) / 32), (unsigned)((N + 31) / 32));
    PFSM_CUDA(cudaMemsetAsync(h->info, 0xFF, sizeof(unsigned long long), st));
    if ((rc = copy_mat(h->S, L, S_in, N, N, st))) return rc;
    if ((rc = copy_mat(h->S + (size_t)N * L, L, A, N, N, st))) return rc;
    extract_diag_kernel<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(h->S, L, n, h->gdiag);
    PFSM_CUDA(cudaGetLastError());
    if ((rc = stacked_cholesky(h, true, st))) return rc;                       // O = [L ; A L^-T]
    transpose_kernel<<<tg, tb, 0, st>>>(h->O + (size_t)N * L, L, h->S + (size_t)N * L, L, n, n);  // (A L^-T)^T = L^-1 A
    PFSM_CUDA(cudaGetLastError());
    if ((rc = stacked_cholesky(h, false, st))) return rc;                      // O bottom = L^-1 A L^-T
    symmetrize_kernel<<<tg, tb, 0, st>>>(h->O + (size_t)N * L, L, Ap_out, ldo, n);
    PFSM_CUDA(cudaGetLastError());
    transpose_kernel<<<tg, tb, 0, st>>>(h->O, L, h->LT, L, n, n);
    PFSM_CUDA(cudaGetLastError());
    transpose_blocks_kernel<<<dim3(4, 4, (unsigned)h->nblk), tb, 0, st>>>(h->Dinv, h->DinvT);
    PFSM_CUDA(cudaGetLastError());
    return 0;
}

// X = L^-T V, in the row-major view X_rm = V_rm L^-1: block back-substitution from the last panel to the first,
// X_k = R_k L_kk^-1, then R[:, c] -= X_k L[k, c] for the column blocks c < k.  All in place in V: the tile that forms
// X_k[r] reads exactly the block R_k[r] it overwrites (every read of the main loop precedes the epilogue's stores), and
// column block k is not touched again, so no second matrix and no final copy are needed.
static int run_generalized_back(pfsm_ctx* h, double* V, cudaStream_t st) {
    const int64_t N = h->N, L = h->ld;
    const int32_t n = (int32_t)N;
    int rc;
    CUtensorMap mapV;
    if ((rc = make_map(&mapV, V, N, N, L))) return rc;
    for (int32_t k = h->nblk - 1; k >= 0; --k) {
        const int32_t k0 = k * CHOL_NB, nb = (int32_t)std::min<int64_t>(CHOL_NB, N - k0);
        GemmParams pp = base_params();
        pp.C = V; pp.ldc = L; pp.cr0 = 0; pp.cc0 = k0; pp.mr = n; pp.nc = nb;
        pp.xr0 = 0; pp.xk0 = k0; pp.yr0 = k * CHOL_NB; pp.yk0 = 0; pp.klen = nb;
        if ((rc = launch_gemm<EPI_PLAIN>(h, mapV, h->mapDT, mapV, pp, st))) return rc;
        if (k0 > 0) {
            GemmParams pt = base_params();
            pt.C = V; pt.ldc = L; pt.cr0 = 0; pt.cc0 = 0; pt.mr = n; pt.nc = k0;
            pt.xr0 = 0; pt.xk0 = k0; pt.yr0 = 0; pt.yk0 = k0; pt.klen = nb;
            if ((rc = launch_gemm<EPI_SUB>(h, mapV, h->mapLT, mapV, pt, st))) return rc;
        }
    }
    return 0;
}

int pfsm_generalized_reduce(pfsm_handle_t h, const double* A, const double* S, double* Ap_out, void* stream) {
    if (!h) return -1;
    if (int rc_dev = check_device(h)) return rc_dev;
    if (!A || ((uintptr_t)A & 7)) return -2;
    if (!S || ((uintptr_t)S & 7)) return -3;
    if (!Ap_out || ((uintptr_t)Ap_out & 7)) return -4;
    int rc;
    if ((rc = ensure_generalized(h))) return rc;
    h->ev_valid = false;
    return run_generalized_reduce(h, A, S, Ap_out, h->N, (cudaStream_t)stream);
}

int pfsm_solve_generalized(pfsm_handle_t h, const double* A, const double* S, double* X_out, double* lambda_out,
                           void* stream) {
    if (!h) return -1;
    if (int rc_dev = check_device(h)) return rc_dev;
    if (!A || ((uintptr_t)A & 7)) return -2;
    if (!S || ((uintptr_t)S & 7)) return -3;
    if (!X_out || ((uintptr_t)X_out & (h->ld == h->N ? 15 : 7))) return -4;
    if (!lambda_out || ((uintptr_t)lambda_out & 7)) return -5;
    int rc;
    if ((rc = ensure_generalized(h))) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    double* Xu;
    if ((rc = stage_in(h, X_out, &h->padV, &Xu, st, false))) return rc;
    if ((rc = run_generalized_reduce(h, A, S, h->Ap, h->ld, st))) return rc;
    // the reduction's status (S not positive definite) must survive the solve's own reset of info
    h->keep_info = true;
    rc = solve_core(h, h->Ap, Xu, lambda_out, stream, 5, nullptr, nullptr);
    h->keep_info = false;
    if (rc) return rc;
    if ((rc = run_generalized_back(h, Xu, st))) return rc;
    return stage_out(h, Xu, X_out, st);
}

// ---- SCF-sequence mode: A is the subspace matrix of a step whose solution is close to the
// previous one.  With the previous eigenvectors V_prev (orthonormal), A' = V_prev^T A V_prev is diagonally dominant
// -- the method's condition for success -- so PFSM runs on A' and the result is rotated back: V = V_prev U. ----
int pfsm_solve_warm(pfsm_handle_t h, const double* A, double* V_inout, double* lambda_out, void* stream) {
    if (!h) return -1;
    if (int rc_dev = check_device(h)) return rc_dev;
    const uintptr_t am = (h->ld == h->N) ? 15 : 7;
    if (!A || ((uintptr_t)A & am)) return -2;
    if (!V_inout || ((uintptr_t)V_inout & am)) return -3;
    if (!lambda_out || ((uintptr_t)lambda_out & 7)) return -4;
    int rc;
    if ((rc = ensure_generalized(h))) return rc;  // Ap and LT double as A' and V_prev^T
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t N = h->N, L = h->ld;
    const int32_t n = (int32_t)N;
    if (!h->Ub && (rc = dev_alloc(h, (void**)&h->Ub, (size_t)N * L * sizeof(double)))) return rc;  // U of the rotated problem
    double *Au, *Vu;
    if ((rc = stage_in(h, A, &h->padA, &Au, st))) return rc;
    if ((rc = stage_in(h, V_inout, &h->padV, &Vu, st))) return rc;
    CUtensorMap mapA, mapV, mapU;
    if ((rc = make_map(&mapA, Au, N, N, L))) return rc;
    if ((rc = make_map(&mapV, Vu, N, N, L))) return rc;
    if ((rc = make_map(&mapU, h->Ub, N, N, L))) return rc;
    const dim3 tb(32, 8), tg((unsigned)((N + 31) / 32), (unsigned)((N + 31) / 32));
    {   // W = V_prev A  (row-major view: row i = (A v_i)^T)
        GemmParams p = base_params();
        p.C = h->W; p.ldc = L; p.mr = n; p.nc = n; p.klen = n;
        if ((rc = launch_gemm<EPI_PLAIN>(h, mapV, mapA, h->mapW, p, st))) return rc;
    }
    {   // A'[i][j] = v_i . (A v_j), into S's top half, then symmetrized into Ap
        GemmParams p = base_params();
        p.C = h->S; p.ldc = L; p.mr = n; p.nc = n; p.klen = n;
        if ((rc = launch_gemm<EPI_PLAIN>(h, mapV, h->mapW, h->mapS, p, st))) return rc;
        symmetrize_kernel<<<tg, tb, 0, st>>>(h->S, L, h->Ap, L, n);
        PFSM_CUDA(cudaGetLastError());
    }
    transpose_kernel<<<tg, tb, 0, st>>>(Vu, L, h->LT, L, n, n);  // V_prev^T, K-contiguous for the rotation back
    PFSM_CUDA(cudaGetLastError());
    if ((rc = solve_core(h, h->Ap, h->Ub, lambda_out, stream, 5, nullptr, nullptr))) return rc;  // U, lambda
    {   // V = V_prev U: row i of the result = sum_k U[i][k] V_prev[k][:], written over V_prev (LT keeps its transpose)
        GemmParams p = base_params();
        p.C = Vu; p.ldc = L; p.mr = n; p.nc = n; p.klen = n;
        if ((rc = launch_gemm<EPI_PLAIN>(h, mapU, h->mapLT, mapV, p, st))) return rc;
    }
    return stage_out(h, Vu, V_inout, st);
}

// ---- f2: the paper's own generalized -> standard conversion (Eq. 14-15; reading R19):
//      Z_0 = A (the identity approximates B^-1),  Z_{n+1} = Z_n - D^-1 (B Z_n - A),  D = diag(B).
// Columns of Z are independent (one block of N/P columns per node in the paper); here all N columns are one
// GEMM per iteration with the update fused in the epilogue.  Works on Y = Z^T (A, B symmetric):
//      Y_{n+1}[j][i] = Y_n[j][i] - (sum_k Y_n[j][k] B[i][k] - A[j][i]) / B[i][i].
int pfsm_standard_form_eq14(pfsm_handle_t h, const double* A, const double* B, double* Z_out, int32_t niter,
                            int32_t symmetrize, void* stream) {
    if (!h) return -1;
    if (int rc_dev = check_device(h)) return rc_dev;
    const uintptr_t am = (h->ld == h->N) ? 15 : 7;
    if (!A || ((uintptr_t)A & am)) return -2;
    if (!B || ((uintptr_t)B & am)) return -3;
    if (!Z_out || ((uintptr_t)Z_out & 7)) return -4;
    if (niter < 0) return -5;
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t N = h->N, L = h->ld;
    const int32_t n = (int32_t)N;
    int rc;
    double *Au, *Bu;
    if ((rc = stage_in(h, A, &h->padA, &Au, st))) return rc;
    if ((rc = stage_in(h, B, &h->padB, &Bu, st))) return rc;
    CUtensorMap mapB;
    if ((rc = make_map(&mapB, Bu, N, N, L))) return rc;
    inv_diag_kernel<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(B, N, n, h->gdiag);
    PFSM_CUDA(cudaGetLastError());
    double* cur = h->W;       // Y_n
    double* nxt = h->S;       // Y_{n+1} (top half of S)
    const CUtensorMap* mcur = &h->mapW;
    const CUtensorMap* mnxt = &h->mapS;
    if ((rc = copy_mat(cur, L, A, N, N, st))) return rc;
    for (int it = 0; it < niter; ++it) {
        GemmParams p = base_params();
        p.C = nxt; p.ldc = L; p.mr = n; p.nc = n; p.klen = n;
        p.E1 = Au; p.ld1 = L; p.E2 = cur; p.ld2 = L; p.eps = h->gdiag;
        if ((rc = launch_gemm<EPI_JSTEP>(h, *mcur, mapB, *mnxt, p, st))) return rc;
        std::swap(cur, nxt);
        std::swap(mcur, mnxt);
    }
    if (symmetrize) {
        const dim3 tb(32, 8), tg((unsigned)((N + 31) / 32), (unsigned)((N + 31) / 32));
        symmetrize_kernel<<<tg, tb, 0, st>>>(cur, L, Z_out, N, n);   // (Y + Y^T)/2 = (Z + Z^T)/2
    } else {
        // column-major Z is the same memory as row-major Y = Z^T
        if ((rc = copy_mat(Z_out, N, cur, L, N, st))) return rc;
    }
    PFSM_CUDA(cudaGetLastError());
    return 0;
}

// ---- f3: one solve sharded over `world` GPUs (the paper's own decomposition, PAPER.md:88,
// 185).  Rank g owns the slices [g P/G, (g+1) P/G), i.e. rows [r0, r1) of the row-major V.  Steps 2-3 and 5 need
// no communication; step 4 needs the vectors of all ranks.  The library provides the four compute phases; the
// caller (paper_1502_07806_b200/sharded.py) runs an all-gather between them:
//   phase 1: steps 2-3 on the own rows of V                       -> all-gather V rows
//   phase 2: own block row of G = V V^T (row-major view)           -> all-gather G rows   (buffer 0)
//   phase 3: Cholesky of G (replicated, N^3/3) + triangular solve of the own rows of V^T (N^3/G)
//                                                                  -> all-gather rows of V^T R^-1 (buffer 1)
//   phase 4: V = (V^T R^-1)^T, step 5 on the own rows              -> all-gather lambda
// copies count doubles at src into buffer `which` of every peer, at element offset `off` of that buffer
static int peer_copy(pfsm_ctx* h, int which, const double* src, size_t off, int64_t count, cudaStream_t st) {
    PeerPtrs d;
    d.n = h->npeer;
    for (int i = 0; i < GEMM_MAX_PEERS; ++i) d.p[i] = i < h->npeer ? h->peer_buf[which][i] + off : nullptr;
    const int blocks = (int)std::min<int64_t>((count + 255) / 256, (int64_t)h->sms * 8);
    peer_copy_kernel<<<blocks, 256, 0, st>>>(src, count, d);
    PFSM_CUDA(cudaGetLastError());
    return 0;
}

int pfsm_set_shard(pfsm_handle_t h, int32_t rank, int32_t world) {
    if (!h) return -1;
    if (world < 1 || (h->N & 1) || h->N % h->P != 0 || h->P % world != 0 || (h->N / world) % BM != 0) return -3;
    if (rank < 0 || rank >= world) return -2;
    h->sh_rank = rank;
    h->sh_world = world;
    h->npeer = 0;
    memset(h->peer_buf, 0, sizeof(h->peer_buf));
    return 0;
}

int pfsm_shard_buffer(pfsm_handle_t h, int32_t which, double** ptr) {
    if (!h) return -1;
    if (!ptr) return -3;
    if (which == 0) *ptr = h->S;                                   // G: N x N (row block = own rows)
    else if (which == 1) *ptr = h->O + (size_t)h->N * h->ld;       // V^T R^-1: N x N (row block = own components)
    else return -2;
    return 0;
}

int pfsm_shard_phase(pfsm_handle_t h, int32_t phase, const double* A, double* V, double* lambda_out, void* stream) {
    if (!h) return -1;
    if (int rc_dev = check_device(h)) return rc_dev;
    if (phase < 1 || phase > 4) return -2;
    if ((phase == 1 || phase == 4) && (!A || ((uintptr_t)A & 15))) return -3;
    if (!V || ((uintptr_t)V & 15)) return -4;
    if (phase == 4 && !lambda_out) return -5;
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t N = h->N, L = h->ld;
    const int32_t n = (int32_t)N;
    const int32_t rows = n / h->sh_world, r0 = h->sh_rank * rows;
    const int32_t ns = h->P / h->sh_world, s0 = h->sh_rank * ns;
    int rc;
    CUtensorMap mapA, mapV;
    if ((rc = make_map(&mapV, V, N, N, L))) return rc;
    if (A && (rc = make_map(&mapA, A, N, N, L))) return rc;
    const dim3 tb(32, 8), tg((unsigned)((N + 31) / 32), (unsigned)((N + 31) / 32));
    h->ev_valid = false;
    if (phase == 1) {
        PFSM_CUDA(cudaMemsetAsync(h->info, 0xFF, sizeof(unsigned long long), st));
        PFSM_CUDA(cudaMemsetAsync(V + (size_t)r0 * N, 0, (size_t)rows * N * sizeof(double), st));
        if ((rc = launch_jacobi(h, A, V, st, s0, ns))) return rc;
        if ((rc = run_step3(h, mapV, mapA, V, r0, rows, st, nullptr, true))) return rc;
        if (h->npeer > 0 && h->iters == 0 && (rc = peer_copy(h, 0, V + (size_t)r0 * L, (size_t)r0 * L, (int64_t)rows * L, st))) return rc;
    } else if (phase == 2) {
        GemmParams p = base_params();  // G[r0:r1, :] = V[r0:r1, :] V^T
        p.C = h->S; p.ldc = L; p.cr0 = r0; p.mr = rows; p.nc = n; p.xr0 = r0; p.klen = n;
        if (h->npeer > 0) {  // ... stored into every rank's G as the tiles finish
            p.npeer = h->npeer;
            for (int i = 0; i < h->npeer; ++i) p.peerC[i] = h->peer_buf[1][i];
            if ((rc = launch_gemm<EPI_PLAIN, true>(h, mapV, mapV, h->mapS, p, st))) return rc;
        } else if ((rc = launch_gemm<EPI_PLAIN>(h, mapV, mapV, h->mapS, p, st))) return rc;
    } else if (phase == 3) {
        transpose_kernel<<<tg, tb, 0, st>>>(V, L, h->S + (size_t)N * L, L, n, n);
        PFSM_CUDA(cudaGetLastError());
        extract_diag_kernel<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(h->S, L, n, h->gdiag);
        PFSM_CUDA(cudaGetLastError());
        if ((rc = stacked_cholesky(h, true, st, r0, r0 + rows, true))) return rc;
    } else {
        transpose_kernel<<<tg, tb, 0, st>>>(h->O + (size_t)N * L, L, V, L, n, n);
        PFSM_CUDA(cudaGetLastError());
        GemmParams p = base_params();
        p.C = h->W; p.ldc = L; p.cr0 = r0; p.mr = rows; p.nc = n; p.xr0 = r0; p.klen = n;
        if ((rc = launch_gemm<EPI_PLAIN>(h, mapV, mapA, h->mapW, p, st))) return rc;
        if ((rc = launch_rayleigh(h, V, lambda_out, r0, rows, st))) return rc;
        if (h->npeer > 0) {
            if ((rc = peer_copy(h, 3, lambda_out + r0, (size_t)r0, rows, st))) return rc;
            if ((rc = peer_copy(h, 4, h->resid + r0, (size_t)r0, rows, st))) return rc;
        }
    }
    return 0;
}

// ---- Peer-write mode of the sharded solve: instead of all-gathering after each phase, every rank stores its share of
// a phase's result straight into the other ranks' buffers -- from the epilogue of the GEMM that produces it
// (gemm_tn_kernel<EPI, true>), tile by tile over NVLink / NVSwitch -- and the ranks only synchronize between phases.
// The other ranks' buffers are ordinary device allocations of their processes, mapped here through CUDA IPC:
//   pfsm_ipc_export  (owner)  handle + byte offset of a device pointer inside its allocation
//   pfsm_ipc_open    (peer)   maps the allocation (lazily enabling peer access) and returns base and pointer
//   pfsm_set_shard_peers      registers, per buffer, the world - 1 mapped pointers of the other ranks
int pfsm_ipc_export(const void* dev_ptr, void* handle64, int64_t* offset) {
    if (!dev_ptr) return -1;
    if (!handle64) return -2;
    if (!offset) return -3;
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "handle size");
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    PFSM_CUDA(cudaGetDriverEntryPoint("cuMemGetAddressRange", &fn, cudaEnableDefault, &q));
    if (q != cudaDriverEntryPointSuccess || !fn) return PFSM_CUDA_ERROR_BASE + (int)cudaErrorNotSupported;
    CUdeviceptr base = 0;
    size_t size = 0;
    if (((CUresult(*)(CUdeviceptr*, size_t*, CUdeviceptr))fn)(&base, &size, (CUdeviceptr)dev_ptr) != CUDA_SUCCESS)
        return PFSM_CUDA_ERROR_BASE + (int)cudaErrorInvalidValue;
    cudaIpcMemHandle_t hd;
    PFSM_CUDA(cudaIpcGetMemHandle(&hd, (void*)base));
    memcpy(handle64, &hd, 64);
    *offset = (int64_t)((CUdeviceptr)dev_ptr - base);
    return 0;
}

int pfsm_ipc_open(const void* handle64, int64_t offset, void** base_out, void** ptr_out) {
    if (!handle64) return -1;
    if (offset < 0) return -2;
    if (!base_out) return -3;
    if (!ptr_out) return -4;
    cudaIpcMemHandle_t hd;
    memcpy(&hd, handle64, 64);
    void* base = nullptr;
    PFSM_CUDA(cudaIpcOpenMemHandle(&base, hd, cudaIpcMemLazyEnablePeerAccess));
    *base_out = base;
    *ptr_out = (char*)base + offset;
    return 0;
}

int pfsm_ipc_close(void* base) {
    if (!base) return -1;
    PFSM_CUDA(cudaIpcCloseMemHandle(base));
    return 0;
}

int pfsm_set_shard_peers(pfsm_handle_t h, int32_t which, void* const* peer_ptrs, int32_t npeer) {
    if (!h) return -1;
    if (which < 0 || which > 4) return -2;
    if (npeer < 0 || npeer > GEMM_MAX_PEERS || npeer != (npeer ? h->sh_world - 1 : 0)) return -4;
    if (npeer > 0 && !peer_ptrs) return -3;
    for (int i = 0; i < npeer; ++i)
        if (!peer_ptrs[i] || ((uintptr_t)peer_ptrs[i] & 7)) return -3;
    for (int i = 0; i < GEMM_MAX_PEERS; ++i) h->peer_buf[which][i] = i < npeer ? (double*)peer_ptrs[i] : nullptr;
    // peer-write mode is on once all five buffers are registered (and off again when any is cleared)
    int32_t all = h->sh_world - 1;
    for (int b = 0; b < 5; ++b)
        for (int i = 0; i < h->sh_world - 1; ++i)
            if (!h->peer_buf[b][i]) all = 0;
    h->npeer = all;
    return 0;
}

int pfsm_solve(pfsm_handle_t h, const double* A, double* V_inout, double* lambda_out, void* stream) {
    return pfsm_solve_partial(h, A, V_inout, lambda_out, stream, 5);
}

// A = A^T: only the lower block triangle (256-row blocks, each with its columns up to the end of its diagonal block)
// crosses PCIe, 52 % of 8 N^2 bytes at N = 8192; the upper part is mirrored on the device (0.2 ms).
static int upload_symmetric(pfsm_ctx* h, const double* A_host, cudaStream_t s) {
    const int64_t N = h->N, L = h->ld, RB = 256;
    for (int64_t r0 = 0; r0 < N; r0 += RB) {
        const int64_t rows = std::min<int64_t>(RB, N - r0), width = std::min<int64_t>(N, r0 + RB);
        PFSM_CUDA(cudaMemcpy2DAsync(h->A_stage + (size_t)r0 * L, (size_t)L * sizeof(double), A_host + (size_t)r0 * N,
                                    (size_t)N * sizeof(double), (size_t)width * sizeof(double), (size_t)rows,
                                    cudaMemcpyHostToDevice, s));
    }
    const dim3 tb(32, 8), tg((unsigned)((N + 31) / 32), (unsigned)((N + 31) / 32));
    mirror_lower_kernel<<<tg, tb, 0, s>>>(h->A_stage, L, (int32_t)N, (int32_t)RB);
    PFSM_CUDA(cudaGetLastError());
    return 0;
}

int pfsm_solve_host(pfsm_handle_t h, const double* A_host, double* V_host, double* lambda_host, void* stream) {
    if (!h) return -1;
    if (int rc_dev = check_device(h)) return rc_dev;
    if (!A_host) return -2;
    if (!V_host) return -3;
    if (!lambda_host) return -4;
    const size_t n2 = (size_t)h->N * h->ld * sizeof(double);
    if (!h->A_stage) {
        int rc;
        if ((rc = dev_alloc(h, (void**)&h->A_stage, n2))) return rc;
        if ((rc = dev_alloc(h, (void**)&h->V_stage, n2))) return rc;
        if ((rc = dev_alloc(h, (void**)&h->lam_stage, h->N * sizeof(double)))) return rc;
    }
    cudaStream_t st = (cudaStream_t)stream;
    int rc;
    if (h->jac_cs > 0 || (h->tridiag && 2 * (size_t)h->P * h->M * h->M <= (size_t)h->N * h->N)) {
        // Step 2 only needs the P diagonal blocks: upload those first (packed, into the workspace the shared-memory
        // Jacobi leaves free and the tridiagonal route works in) and let the full matrix follow on the side stream
        // under the step-2 kernels.  (Not when the blocks are as large as A itself: wide windows.)
        const size_t M = (size_t)h->M;
        for (int32_t sl = 0; sl < h->P; ++sl) {
            const int64_t lo = h->tab_host[(size_t)h->P + sl];
            PFSM_CUDA(cudaMemcpy2DAsync(h->Gws + (size_t)sl * M * M, M * sizeof(double), A_host + (size_t)lo * h->N + lo,
                                        (size_t)h->N * sizeof(double), M * sizeof(double), M, cudaMemcpyHostToDevice, st));
        }
        PFSM_CUDA(cudaEventRecord(h->ev_fork, st));
        PFSM_CUDA(cudaStreamWaitEvent(h->side, h->ev_fork, 0));
        if ((rc = upload_symmetric(h, A_host, h->side))) return rc;
        PFSM_CUDA(cudaEventRecord(h->ev_rest, h->side));
        rc = solve_core(h, h->A_stage, h->V_stage, h->lam_stage, stream, 4, h->Gws, h->ev_rest);  // steps 2-4: V is final
    } else {
        if ((rc = upload_symmetric(h, A_host, st))) return rc;
        rc = solve_core(h, h->A_stage, h->V_stage, h->lam_stage, stream, 4, nullptr, nullptr);
    }
    if (rc) return rc;
    // V goes back to the host on the side stream while step 5 (which only reads V) computes lambda
    PFSM_CUDA(cudaEventRecord(h->ev_fork, st));
    PFSM_CUDA(cudaStreamWaitEvent(h->side, h->ev_fork, 0));
    PFSM_CUDA(cudaMemcpy2DAsync(V_host, (size_t)h->N * sizeof(double), h->V_stage, (size_t)h->ld * sizeof(double),
                                (size_t)h->N * sizeof(double), (size_t)h->N, cudaMemcpyDeviceToHost, h->side));
    PFSM_CUDA(cudaEventRecord(h->ev_chain, h->side));
    {   // step 5 on the staged (leading dimension ld) matrices
        CUtensorMap mapA, mapV;
        if ((rc = make_map(&mapA, h->A_stage, h->N, h->N, h->ld))) return rc;
        if ((rc = make_map(&mapV, h->V_stage, h->N, h->N, h->ld))) return rc;
        h->ev_valid = false;
        if ((rc = run_step5(h, mapV, mapA, h->V_stage, h->lam_stage, st))) return rc;
    }
    PFSM_CUDA(cudaMemcpyAsync(lambda_host, h->lam_stage, h->N * sizeof(double), cudaMemcpyDeviceToHost, st));
    PFSM_CUDA(cudaStreamWaitEvent(st, h->ev_chain, 0));  // join: the caller's stream covers both copies
    return 0;
}

int pfsm_get_info(pfsm_handle_t h, void* stream, int64_t* info) {
    if (!h) return -1;
    if (int rc_dev = check_device(h)) return rc_dev;
    if (!info) return -3;
    unsigned long long v = 0;
    PFSM_CUDA(cudaMemcpyAsync(&v, h->info, sizeof(v), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    PFSM_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
    // (the step-2 kernels form their code from the leading dimension: ld + s + 1)
    *info = (v == ULLONG_MAX) ? 0 : ((int64_t)v > h->ld ? (int64_t)v - (h->ld - h->N) : (int64_t)v);
    return 0;
}

int pfsm_check_validity(pfsm_handle_t h, void* stream, double resid_tol, int32_t* use_standard_solver,
                        double* max_resid_out, int64_t* info_out) {
    if (!h) return -1;
    if (int rc_dev = check_device(h)) return rc_dev;
    if (!(resid_tol >= 0.0)) return -3;
    if (!use_standard_solver) return -4;
    cudaStream_t st = (cudaStream_t)stream;
    // gdiag (step 4's scratch) is free after a solve: slot 0 receives the maximum
    max_residual_kernel<<<1, 1024, 0, st>>>(h->resid, h->N, h->gdiag);
    PFSM_CUDA(cudaGetLastError());
    double mx = 0.0;
    unsigned long long v = 0;
    PFSM_CUDA(cudaMemcpyAsync(&mx, h->gdiag, sizeof(double), cudaMemcpyDeviceToHost, st));
    PFSM_CUDA(cudaMemcpyAsync(&v, h->info, sizeof(v), cudaMemcpyDeviceToHost, st));
    PFSM_CUDA(cudaStreamSynchronize(st));
    const int64_t info = (v == ~0ULL) ? 0 : ((int64_t)v > h->ld ? (int64_t)v - (h->ld - h->N) : (int64_t)v);
    *use_standard_solver = (info != 0 || !(mx <= resid_tol)) ? 1 : 0;
    if (max_resid_out) *max_resid_out = mx;
    if (info_out) *info_out = info;
    return 0;
}

int pfsm_get_step2_sweeps(pfsm_handle_t h, void* stream, int32_t* max_sweeps) {
    if (!h) return -1;
    if (int rc_dev = check_device(h)) return rc_dev;
    if (!max_sweeps) return -3;
    std::vector<int> cnt((size_t)h->P * JACOBI_MAX_SWEEPS);
    PFSM_CUDA(cudaMemcpyAsync(cnt.data(), h->rotcnt, cnt.size() * sizeof(int), cudaMemcpyDeviceToHost,
                              (cudaStream_t)stream));
    PFSM_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
    int mx = 0;
    for (int s = 0; s < h->P; ++s) {
        int k = 0;
        while (k < JACOBI_MAX_SWEEPS && cnt[(size_t)s * JACOBI_MAX_SWEEPS + k] != 0) ++k;
        mx = std::max(mx, std::min(k + 1, (int)JACOBI_MAX_SWEEPS));
    }
    *max_sweeps = mx;
    return 0;
}

int pfsm_get_residuals(pfsm_handle_t h, const double** r) {
    if (!h) return -1;
    if (!r) return -2;
    *r = h->resid;
    return 0;
}

int pfsm_get_shifts(pfsm_handle_t h, const double** e) {
    if (!h) return -1;
    if (!e) return -2;
    *e = h->eps;
    return 0;
}

int pfsm_set_cholqr_passes(pfsm_handle_t h, int32_t passes) {
    if (!h) return -1;
    if (passes < 1 || passes > 2) return -2;
    h->cholqr_passes = passes;
    return 0;
}

// Options select among kernels that compute the same thing (A/B measurements; the parity tests reach every kernel through
// them).  Explicit per-handle state: the library reads no environment variable.
int pfsm_set_option(pfsm_handle_t h, const char* key, int64_t value) {
    if (!h) return -1;
    if (!key) return -2;
    auto is01 = [&](int64_t v) { return v == 0 || v == 1; };
    bool relayout = false;
    if (!strcmp(key, "step2_route")) {
        if (value < 0 || value > 3) return -3;
        h->opt_route = (int32_t)value; relayout = true;
    } else if (!strcmp(key, "jacobi_l2")) {
        if (!is01(value)) return -3;
        h->opt_jacobi_l2 = (int32_t)value; relayout = true;
    } else if (!strcmp(key, "jacobi_cluster_size")) {
        if (value != 0 && value != 1 && value != 2 && value != 4 && value != 8) return -3;
        h->opt_jacobi_cs = (int32_t)value; relayout = true;
    } else if (!strcmp(key, "jacobi_full_cta")) {
        if (!is01(value)) return -3;
        h->opt_jacobi_full = (int32_t)value; relayout = true;
    } else if (!strcmp(key, "sytrd_storage")) {
        if (value < 0 || value > 3) return -3;
        h->opt_sytrd_storage = (int32_t)value;
    } else if (!strcmp(key, "sytrd_grid_barrier")) {
        if (value < 0 || value > 2) return -3;
        h->opt_sytrd_grid = (int32_t)value;
    } else if (!strcmp(key, "cholesky_group")) {
        if (value != 0 && value != 2 && value != 4) return -3;
        h->opt_chol_group = (int32_t)value;
    } else if (!strcmp(key, "cholesky_lookahead")) {
        if (!is01(value)) return -3;
        h->lookahead = value != 0;
    } else if (!strcmp(key, "chain_launches")) {
        if (!is01(value)) return -3;
        h->chain = value != 0;
    } else if (!strcmp(key, "cholqr_passes")) {
        if (value < 1 || value > 2) return -3;
        h->cholqr_passes = (int32_t)value;
    } else {
        return -2;
    }
    if (relayout) {
        int rc;
        if ((rc = check_device(h))) return rc;
        choose_jacobi_layout(h);
        if ((rc = ensure_tridiag_ws(h))) return rc;
    }
    return 0;
}

int pfsm_set_alpha(pfsm_handle_t h, double alpha) {
    if (!h) return -1;
    if (!std::isfinite(alpha) || !(alpha > 0.0)) return -2;
    h->alpha = alpha;
    return 0;
}

size_t pfsm_workspace_bytes(pfsm_handle_t h) { return h ? h->bytes : 0; }

int64_t pfsm_launches_per_solve(pfsm_handle_t h) {
    if (!h) return 0;
    // jacobi + 2 iters GEMMs + (2 transposes + Gram + diag extract + per panel: diag, panel, trailing (none after the last)) + GEMM + rayleigh
    {
        const int64_t nb = h->nblk;
        // per panel: chol_diag + panel GEMM; inside a group one inner update per panel after its first; trailing updates: one
        // per group with columns left, split in two (next group's columns / the rest) when the look-ahead schedule is active
        const std::vector<int32_t> gb = chol_group_bounds(h);
        const int64_t ngroups = (int64_t)gb.size() - 1;
        int64_t trailing = 0, pairs = 0;  // pairs = inner updates
        for (int64_t g = 0; g < ngroups; ++g) {
            pairs += gb[g + 1] - gb[g] - 1;
            const int64_t cn0 = std::min<int64_t>(h->N, (int64_t)gb[g + 1] * CHOL_NB);
            const int64_t cn1 = std::min<int64_t>(h->N, (int64_t)gb[std::min<size_t>((size_t)g + 2, gb.size() - 1)] * CHOL_NB);
            if (cn0 >= h->N) continue;
            trailing += (h->lookahead && ngroups >= 3 && cn1 < h->N) ? 2 : 1;
        }
        // tridiagonal route: tridiagonalization, bisection, inverse iteration, cluster pass, back-transformation; the blocked
        // tridiagonalization is a copy, one panel kernel per 32 columns and one trailing update per panel but the last
        int64_t step2 = h->tridiag ? 5 : 1;
        if (uses_blocked_sytrd(h, h->P)) {
            const int64_t panels = (h->M - 1 + SB_NB - 1) / SB_NB, waves = (h->P + h->sms - 1) / h->sms;
            int64_t gemms = 0;
            for (int64_t k0 = 0; k0 < h->M - 1; k0 += SB_NB) gemms += (k0 + SB_NB < h->M - 1) ? 1 : 0;
            step2 = 4 + 1 + waves * (panels + gemms);
        }
        return step2 + 2 * (int64_t)h->iters + h->cholqr_passes * (2 + 1 + 1 + 2 * nb + pairs + trailing) + 2;
    }
}

int pfsm_enable_step_timing(pfsm_handle_t h, int32_t enable) {
    if (!h) return -1;
    h->timing = enable != 0;
    h->ev_valid = false;
    return 0;
}

int pfsm_get_step_ms(pfsm_handle_t h, float* ms4) {
    if (!h) return -1;
    if (!ms4) return -2;
    if (!h->ev_valid) return -1;
    PFSM_CUDA(cudaEventSynchronize(h->ev[4]));
    for (int i = 0; i < 4; ++i) PFSM_CUDA(cudaEventElapsedTime(&ms4[i], h->ev[i], h->ev[i + 1]));
    return 0;
}

int pfsm_probe_fp64_peak(int32_t kind, void* stream, double* tflops) {
    if (kind < 0 || kind > 1) return -1;
    if (!tflops) return -3;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    PFSM_CUDA(cudaGetDevice(&dev));
    PFSM_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double* sink = nullptr;
    PFSM_CUDA(cudaMalloc(&sink, 8));
    cudaEvent_t e0, e1;
    PFSM_CUDA(cudaEventCreate(&e0));
    PFSM_CUDA(cudaEventCreate(&e1));
    const int blocks = sms * 4, threads = 256;
    const int iters = (kind == 0) ? 20000 : 40000;
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        PFSM_CUDA(cudaEventRecord(e0, st));
        if (kind == 0)
            probe_dmma_kernel<<<blocks, threads, 0, st>>>(iters, sink);
        else
            probe_dfma_kernel<<<blocks, threads, 0, st>>>(iters, sink);
        PFSM_CUDA(cudaEventRecord(e1, st));
        PFSM_CUDA(cudaEventSynchronize(e1));
        float ms = 0;
        PFSM_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && ms < best) best = ms;
    }
    // per warp per iteration: DMMA 16 x (8*8*4*2) flops; DFMA 16 x 32 x 2 flops
    const double per_warp_iter = (kind == 0) ? 16.0 * 512.0 : 16.0 * 64.0;
    const double flops = per_warp_iter * (double)iters * (threads / 32) * (double)blocks;
    *tflops = flops / ((double)best * 1e-3) * 1e-12;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    return 0;
}

// ---- Allocation-free step 5 (reading R11): lambda_i = v_i^T A v_i, r_i = ||A v_i - lambda_i v_i||_2 for callers that cannot
// call cudaMalloc (CUDA graph capture, tight serving loops, harnesses that forbid it).  No handle (pfsm_create allocates):
// the N x N product T = V A goes to the file-scope static device array above, everything else is the caller's.  Same two
// kernels as pfsm_rayleigh (gemm_tn_kernel<PLAIN>, rayleigh_kernel), same operation order, same bits.  Calls no cudaMalloc,
// cudaFree or allocating library routine.  T is overwritten in full before it is read, so nothing has to be cleared between
// calls; every call on a device shares the one array, so calls that overlap on the GPU (different streams) race.
int pfsm_rayleigh_noalloc(int64_t N, const double* A, const double* V, double* lambda_out, double* resid_out, void* stream) {
    if (N < 2 || (N & 1) || N > PFSM_NOALLOC_MAX_N) return PFSM_ERR_NOALLOC_SIZE;
    if (!A || ((uintptr_t)A & 15)) return -2;
    if (!V || ((uintptr_t)V & 15)) return -3;
    if (!lambda_out || ((uintptr_t)lambda_out & 7)) return -4;
    if (!resid_out || ((uintptr_t)resid_out & 7)) return -5;
    cudaStream_t st = (cudaStream_t)stream;
    double* T = nullptr;
    int rc;
    if ((rc = noalloc_scratch_ptr(&T))) return rc;
    CUtensorMap mapA, mapV, mapT;
    if ((rc = make_map(&mapA, A, N, N, N))) return rc;
    if ((rc = make_map(&mapV, V, N, N, N))) return rc;
    if ((rc = make_map(&mapT, T, N, N, N))) return rc;
    pfsm_ctx launch_state;  // on the stack: only launch_gemm's per-handle flags are used (no workspace, no allocation)
    launch_state.N = N;
    launch_state.ld = N;
    GemmParams p = base_params();
    p.C = T; p.ldc = N; p.mr = (int32_t)N; p.nc = (int32_t)N; p.klen = (int32_t)N;
    if ((rc = launch_gemm<EPI_PLAIN>(&launch_state, mapV, mapA, mapT, p, st))) return rc;
    rayleigh_kernel<<<(unsigned)N, RAY_THREADS, 0, st>>>(V, T, N, N, lambda_out, resid_out, 0);
    PFSM_CUDA(cudaGetLastError());
    return 0;
}

}  // extern "C"
