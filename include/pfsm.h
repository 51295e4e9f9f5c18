/*
 * pfsm.h -- C ABI of libpfsm: one partitioned-folded-spectrum-method (PFSM) solve of the dense
 * real-symmetric FP64 eigenproblem  A V = V Lambda  on one NVIDIA B200 (sm_100a).
 *
 * Method: E.L. Briggs, C.T. Kelley, J. Bernholc, "Parallel implementation of electronic structure
 * eigensolver using a partitioned folded spectrum method", arXiv:1502.07806, section II
 * (PAPER.md:47-100).  The interface follows the paper's stated intent, "a separate library with a
 * calling interface similar to the standard eigensolvers" (section VI): LAPACK-like,
 * column-major, integer status codes.
 *
 * The five steps one solve runs, all in hand-written CUDA kernels on the caller's stream:
 *   1. partition   N eigenpairs -> P contiguous slices of m = N/P; slice s owns the principal
 *                  submatrix B_s = A[lo:lo+M, lo:lo+M], M = min(N, m + 2*window),
 *                  lo = clamp(s*m - window, 0, N - M)                      (Fig. 1)
 *   2. submatrix   batched symmetric eigensolve B_s y = mu y; the slice's m eigenpairs (local
 *      eigensolve  ascending indices s*m-lo .. s*m-lo+m-1) give shifts eps_i = mu and zero-padded
 *                  start vectors x_i^0
 *   3. folded      iters times:  x_i <- x_i - alpha (A - eps_i I)^2 x_i, applied as two successive
 *      spectrum    products W = A V - V diag(eps), V <- V - alpha (A W - W diag(eps))
 *                                                                  (Eq. 5 and 11)
 *   4. Gram-       all N vectors, ascending column order, done as Cholesky-QR:
 *      Schmidt     G = V^T V = R^T R, V <- V R^-1
 *   5. eigenvalues lambda_i = v_i^T A v_i and r_i = ||A v_i - lambda_i v_i||_2 (the paper does not
 *                  say how lambda is produced after step 4; Rayleigh quotients are this library's reading)
 *
 * Conventions common to every call
 *   - All matrices are FP64, column-major with leading dimension N.  Eigenvector i is the
 *     contiguous column V + i*N.  A is full storage: both triangles valid and exactly mirrored.
 *   - "device" pointers are CUDA device memory on the device current at pfsm_create; "host"
 *     pointers are ordinary (ideally pinned) host memory.  Device matrices must be 16-byte aligned (8 for odd N).
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  pfsm_solve
 *     only enqueues work and returns without synchronizing the host.
 *   - Return value: 0 = success; -k = the k-th argument is invalid (LAPACK convention);
 *     >= 1000 = 1000 + cudaError_t of a failed CUDA call.  Numerical status is reported separately
 *     and asynchronously through pfsm_get_info.
 *   - The library never frees or reallocates caller memory and never modifies A.  The handle owns
 *     its workspace.  One handle = one solve in flight; handles are not thread-safe; distinct
 *     handles on distinct streams are independent.
 *   - There is no CPU fallback: every call fails with a CUDA error code if no sm_100 device is usable.
 */
#ifndef PFSM_H
#define PFSM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pfsm_ctx* pfsm_handle_t; /* opaque */

#define PFSM_CUDA_ERROR_BASE 1000

/*
 * Create a solver for fixed (N, P, window, iters, alpha) and allocate its device workspace
 * (about 5 N^2 doubles + P M^2 doubles) on the current device.           [step 1, PAPER.md:88]
 *   out     host pointer receiving the handle
 *   N       matrix order; N >= 2.  Odd N is accepted: tensor maps need a 16-byte row pitch, so internal matrices use the
 *           leading dimension N + 1 and the caller's matrices (leading dimension N, 8-byte alignment suffices) are staged
 *           through padded copies (two extra N^2 device buffers, two extra 2-D copies per call); even N runs in place.
 *           pfsm_set_shard needs an even N.
 *   P       number of spectral slices; 1 <= P <= N.  Slice s holds eigen-indices floor(s N / P) .. floor((s+1) N / P) - 1:
 *           N/P of them when P divides N (the paper writes m = N/P), else floor(N/P) or ceil(N/P) (reading R14)
 *   window  halo rows/columns added on each side of a slice's diagonal block; >= 0.
 *           M = min(N, ceil(N/P) + 2*window), the order of every submatrix, must be <= 8192 in this version (else -4; the
 *           paper ran "M <= 3000"; 4096 < M <= 8192 always takes the lower-triangle tridiagonalization).  Step 2 is a Householder tridiagonalization + multi-section + inverse
 *           iteration (with re-orthogonalization inside tight eigenvalue clusters) + back-transformation of the slice's own
 *           eigenpairs: the submatrix resident in its cluster's distributed shared memory for small M (the BASELINE
 *           configs), L2- or HBM-resident up to the paper's wide windows, gamma = M/N = 0.2-0.3, where
 *           it is blocked with DMMA trailing updates.  A shared-memory cluster Jacobi serves M < 16 and is selectable by
 *           pfsm_set_option.  All routes deliver the eigenpairs to O(eps ||B||).
 *   iters   folded-spectrum iterations of Eq. 11; >= 0
 *   alpha   step length of Eq. 11; finite and > 0.  The library does not estimate spectra:
 *           alpha = 0.5 / max|lambda|^2 keeps every damping factor 1 - alpha (lambda - eps)^2 in [-1, 1].
 * Errors: -1..-6 for the corresponding argument; 1000+cudaError on allocation failure.
 * A handle belongs to the device that was current at pfsm_create: every later call that enqueues work returns
 * 1000+cudaErrorInvalidDevice if another device is current.  Handles on different devices (or streams) are independent;
 * no state is shared between handles.
 */
int pfsm_create(pfsm_handle_t* out, int64_t N, int32_t P, int32_t window, int32_t iters, double alpha);

/*
 * Enqueue one PFSM solve (steps 2-5) on `stream`.                         [PAPER.md:86-96]
 *   A          device, N x N, symmetric, read only
 *   V_inout    device, N x N.  On output column i is the i-th orthonormal approximate eigenvector.
 *              Its input content is ignored in this version: start vectors come only from the
 *              submatrix solutions.
 *   lambda_out device, N.  lambda_out[i] belongs to column i (slice order; not re-sorted).
 * Errors: -1 null handle, -2/-3/-4 null or misaligned pointer, 1000+cudaError on launch failure.
 */
int pfsm_solve(pfsm_handle_t h, const double* A, double* V_inout, double* lambda_out, void* stream);

/*
 * Same solve with HOST buffers: copies A host->device, runs pfsm_solve, copies V and lambda back,
 * all asynchronously (pinned host memory recommended), using device staging buffers owned by the handle
 * (2 N^2 doubles more, allocated on first use).  The copies overlap the compute: the P diagonal blocks that
 * step 2 needs go first, the full matrix follows on an internal stream under the step-2 kernel, and V returns
 * while step 5 runs; everything is joined back into `stream`, which the caller synchronizes before reading
 * V_host / lambda_host.  A is symmetric, so only its lower block triangle (256-row blocks, each up to the end of its
 * diagonal block) and the P diagonal submatrices are read from A_host and sent over PCIe; the rest is mirrored on the device.  (pfsm_solve, with a
 * device matrix, reads both triangles: reading R15.)
 */
int pfsm_solve_host(pfsm_handle_t h, const double* A_host, double* V_host, double* lambda_host, void* stream);

/*
 * Diagnostic variant of pfsm_solve that stops after step `last_step` (2, 3, 4 or 5) and leaves V in
 * its state after that step (2: zero-padded start vectors; 3: after the folded-spectrum iterations;
 * 4: orthonormalized; 5 = pfsm_solve).  lambda_out is written only when last_step == 5 and may be
 * NULL otherwise.  Used by the parity tests to compare each step with the oracle.
 */
int pfsm_solve_partial(pfsm_handle_t h, const double* A, double* V_inout, double* lambda_out, void* stream,
                       int32_t last_step);

/*
 * Step 4 alone ("Gram-Schmidt orthogonalization"): orthonormalize the N columns of
 * V_inout (device, N x N) in ascending column order, V <- V R^-1 with V^T V = R^T R.  Resets and sets the
 * handle's info like pfsm_solve (pivot j counts as not positive when it is <= 1e-12 ||v_j||^2).
 */
int pfsm_orthonormalize(pfsm_handle_t h, double* V_inout, void* stream);

/*
 * Step 5 alone: lambda_out[i] = v_i^T A v_i and the handle's residual buffer r_i = ||A v_i - lambda_i v_i||_2
 * for the N columns of V (device, N x N, assumed orthonormal; read only).
 */
int pfsm_rayleigh(pfsm_handle_t h, const double* A, const double* V, double* lambda_out, void* stream);

/*
 * Generalized problem A x = lambda S x (Eq. 13; BASELINE.json configs[4] "generalized form ...
 * reduced by Cholesky(S)").  S = L L^T, A' = L^-1 A L^-T (symmetrized), PFSM steps 2-5 on A', X = L^-T V.
 *   A, S       device, N x N, symmetric, read only; S positive definite
 *   X_out      device, N x N: column i = generalized eigenvector i, X^T S X = I
 *   lambda_out device, N
 * The residual buffer then holds the standard-form residuals ||A' v_i - lambda_i v_i||_2.  info in 1..N can
 * also mean that pivot `info` of Cholesky(S) was not positive.  Allocates 2 N^2 doubles more on first use.
 * pfsm_generalized_reduce runs the reduction alone and writes A' to Ap_out (device, N x N).
 */
int pfsm_solve_generalized(pfsm_handle_t h, const double* A, const double* S, double* X_out, double* lambda_out,
                           void* stream);
int pfsm_generalized_reduce(pfsm_handle_t h, const double* A, const double* S, double* Ap_out, void* stream);

/*
 * SCF-sequence mode ("a sequence of eigenvalue problems where the solution ... is similar but not
 * identical to the solution from the previous iteration"; A must be diagonally dominant).
 * V_inout holds, on input, the ORTHONORMAL eigenvectors V_prev of the previous step (e.g. from the last
 * pfsm_solve_warm, or from a standard eigensolver for the first steps).  The call forms
 * A' = V_prev^T A V_prev, runs steps 2-5 on A', and returns V = V_prev U (orthonormal) and lambda.  Residuals
 * are those of (A, V).  Costs three more N^3 products than pfsm_solve; 2 N^2 doubles more workspace on first use.
 * If get_info != 0 or the residuals are large, A was not close enough to the previous step: fall back to a
 * standard eigensolver for this step.
 */
int pfsm_solve_warm(pfsm_handle_t h, const double* A, double* V_inout, double* lambda_out, void* stream);

/*
 * The paper's own generalized -> standard conversion (section V, Eq. 14-15): Z = B^-1 A by
 * the column-parallel iteration  Z_0 = A,  Z_{n+1} = Z_n - D^-1 (B Z_n - A),  D = diag(B)  (Eq. 14 prints
 * "D^-1 A x"; the matrix iteration is meant), niter times; one fused GEMM per iteration.
 *   A, B    device, N x N, symmetric; B diagonally dominant (the iteration converges iff rho(I - D^-1 B) < 1)
 *   Z_out   device, N x N, column-major.  symmetrize != 0 returns (Z + Z^T)/2, the matrix "used in Eq. (3)";
 *           symmetrize == 0 returns Z itself (not symmetric in general).
 * Compare pfsm_generalized_reduce, which reduces by Cholesky(B) instead.
 */
int pfsm_standard_form_eq14(pfsm_handle_t h, const double* A, const double* B, double* Z_out, int32_t niter,
                            int32_t symmetrize, void* stream);

/*
 * One solve sharded over `world` GPUs (one process and one handle per GPU; the paper's decomposition of slices
 * over nodes, with its all-gather).  Rank g owns slices [g P/world, (g+1) P/world),
 * i.e. columns [g N/world, (g+1) N/world) of V.  Requires N % P == 0, P % world == 0 and (N/world) % 128 == 0.  A is
 * replicated.  pfsm_shard_phase runs compute phase 1..4 on the rank's share; between the phases the CALLER
 * all-gathers (NCCL/torch.distributed; see paper_1502_07806_b200/sharded.py):
 *   after phase 1 (steps 2-3 on own columns):   the column blocks of V                  (V itself, N x N)
 *   after phase 2 (own block of V^T V):          the blocks of pfsm_shard_buffer(h, 0)   (N x N)
 *   after phase 3 (Cholesky + own share of the triangular solve): blocks of pfsm_shard_buffer(h, 1) (N x N)
 *   after phase 4 (V assembled, step 5 on own columns): the blocks of lambda_out (and of the residuals)
 * Every buffer is split into `world` equal contiguous blocks of N/world columns (column-major), rank g's first.
 * A may be NULL in phases 2-3, lambda_out in phases 1-3.  get_info reports as for pfsm_solve.
 */
int pfsm_set_shard(pfsm_handle_t h, int32_t rank, int32_t world);
int pfsm_shard_phase(pfsm_handle_t h, int32_t phase, const double* A, double* V, double* lambda_out, void* stream);
int pfsm_shard_buffer(pfsm_handle_t h, int32_t which, double** device_ptr);

/*
 * PEER-WRITE MODE of the sharded solve: the exchange fused into the kernels that produce the data.  Instead of the caller
 * all-gathering after each phase, every rank stores its share of a phase's result straight into the other ranks' buffers:
 * the GEMM epilogues of phases 1-3 write each finished C tile to all ranks (peer device memory over NVLink / NVSwitch), a
 * small copy kernel does the same for lambda and the residuals.  The caller then only needs a BARRIER between the phases
 * (all ranks' phase-k work complete before anyone starts phase k+1) and one after phase 4 -- the paper's MPI_Allgatherv
 * disappears into the product's own stores.  Results are those of the gather mode, bit for bit.
 *   pfsm_ipc_export   owner process: 64-byte CUDA IPC handle of the allocation that holds `dev_ptr`, and dev_ptr's byte
 *                     offset in it (the handle travels to the other ranks as plain bytes, e.g. by all_gather_object)
 *   pfsm_ipc_open     peer process: maps that allocation (enabling peer access on first use); *base_out is what
 *                     pfsm_ipc_close takes, *ptr_out = base + offset is the usable device pointer
 *   pfsm_set_shard_peers(h, which, peer_ptrs, npeer)   after pfsm_set_shard: the other ranks' buffer `which`
 *                     (0: V, 1: pfsm_shard_buffer 0, 2: pfsm_shard_buffer 1, 3: lambda_out, 4: the residuals), npeer =
 *                     world - 1 mapped pointers in any order (npeer = 0 clears).  The mode is on once all five are set.
 * Every rank must pass the SAME V and lambda_out buffers to pfsm_shard_phase that its peers registered.  world <= 8.
 * Errors: -k for argument k; 1000+cudaError (e.g. the allocation cannot be shared: not from cudaMalloc).
 */
int pfsm_ipc_export(const void* dev_ptr, void* handle64, int64_t* offset);
int pfsm_ipc_open(const void* handle64, int64_t offset, void** base_out, void** ptr_out);
int pfsm_ipc_close(void* base);
int pfsm_set_shard_peers(pfsm_handle_t h, int32_t which, void* const* peer_ptrs, int32_t npeer);

/* Release the handle and its workspace (synchronizes the device).  NULL is a no-op returning 0. */
int pfsm_destroy(pfsm_handle_t h);

/*
 * Numerical status of the last solve; synchronizes `stream` (the stream that solve was enqueued on -- the one argument
 * this call adds to SURVEY.md 8(b)'s proposed signature: the handle does not remember streams, the caller owns them).
 *   *info = 0        success
 *   1 <= *info <= N  Cholesky pivot *info of V^T V was not positive (<= 1e-12 x its original diagonal
 *                    entry): the N vectors are numerically
 *                    dependent -- the paper's failure mode for a matrix that is not diagonally
 *                    dominant.  Outputs are undefined; use a standard eigensolver
 *                    for this step.
 *   *info = N+s+1    the submatrix eigensolver of slice s did not converge within its sweep cap.
 */
int pfsm_get_info(pfsm_handle_t h, void* stream, int64_t* info);

/*
 * The paper's validity guard in one call (PFSM needs a diagonally dominant matrix, "standard
 * diagonalization" is used while that does not hold): after a full solve (pfsm_solve, _host, _warm, _generalized)
 * reduces the residual norms on the device and synchronizes `stream`.
 *   resid_tol            largest acceptable r_i = ||A v_i - lambda_i v_i||_2 (absolute; scale it with ||A||); >= 0
 *   *use_standard_solver host, out: 1 if pfsm_get_info would be non-zero or max_i r_i > resid_tol (NaN counts as
 *                        too large) -- the caller should diagonalize this step with a standard solver -- else 0
 *   *max_resid_out       host, out, optional (may be NULL): max_i r_i
 *   *info_out            host, out, optional: the same value pfsm_get_info returns
 * Errors: -1 handle, -3 resid_tol negative or NaN, -4 NULL verdict pointer, 1000+cudaError.
 */
int pfsm_check_validity(pfsm_handle_t h, void* stream, double resid_tol, int32_t* use_standard_solver,
                        double* max_resid_out, int64_t* info_out);

/* Largest number of Jacobi sweeps any slice's submatrix eigensolve (step 2) used in the last solve;
 * synchronizes `stream`.  The last sweep is the one that found nothing left to rotate.  Reads 1 when step 2 took
 * the tridiagonal route (the default from M = 16 on), which has no sweeps. */
int pfsm_get_step2_sweeps(pfsm_handle_t h, void* stream, int32_t* max_sweeps);

/* Device pointer to the N residual norms r_i = ||A v_i - lambda_i v_i||_2 of the last solve (step 5). */
int pfsm_get_residuals(pfsm_handle_t h, const double** r_device);

/* Device pointer to the N shifts eps_i (submatrix eigenvalues) of the last solve (step 2). */
int pfsm_get_shifts(pfsm_handle_t h, const double** eps_device);

/*
 * Number of Cholesky-QR passes of step 4: 1 (default) or 2.  One pass leaves ||V^T V - I||_max ~ eps cond(V)^2, which
 * meets the 1e-12 N gate up to cond(V) ~ 1e3 (BASELINE config 4: cond ~ 500, 5e-13 measured); a second pass
 * (CholeskyQR2) brings it to ~eps for cond(V) up to ~1e7 at the cost of step 4 twice.  The exact-arithmetic result,
 * the Gram-Schmidt basis in ascending column order, is the same.
 */
int pfsm_set_cholqr_passes(pfsm_handle_t h, int32_t passes);

/*
 * Select among kernels / schedules that compute the same result.  Explicit per-handle state: the library reads no
 * environment variable.  Defaults (all 0 except where noted) are the product path; the other values exist for A/B
 * measurements and so that the parity tests reach every kernel.  Call between solves (not while one is in flight).
 *   key (host C string)      value
 *   "step2_route"            0 auto (M <= 160 shared-memory Jacobi, else tridiagonal route), 1 Jacobi family (M <= 512),
 *                            2 tridiagonal route at any M, 3 persistent-grid Jacobi at any M        [PAPER.md:86-94]
 *   "jacobi_l2"              1: the L2-resident Jacobi kernel instead of the shared-memory one
 *   "jacobi_cluster_size"    0 auto, or 1 | 2 | 4 | 8 CTAs per slice for the shared-memory Jacobi
 *   "jacobi_full_cta"        1: never use the half-CTA layout of the shared-memory Jacobi
 *   "sytrd_storage"          0 auto (full storage while the batch of submatrices fits L2, lower triangle beyond, blocked
 *                            -- panels of 32 columns + one DMMA rank-64 trailing update each -- beyond 1.5 x L2),
 *                            1 full storage, 2 lower triangle, 3 blocked (M even)
 *   "sytrd_grid_barrier"     small M (<= 768): 0 = submatrix resident in the cluster's distributed shared memory when it
 *                            fits (default), 2 = L2-resident submatrix with cluster barriers, 1 = with the grid barrier
 *   "cholesky_lookahead"     default 1; 0: step 4 on one stream                                    [PAPER.md:94-96]
 *   "cholesky_group"         panels (of 128 columns) per trailing update of step 4: 0 auto (4 from N = 6144 on, while more than
 *                            24 panels remain, else 2), 2, 4
 *   "chain_launches"         default 1; 0: the step-3 / step-4 GEMMs in plain stream order (same bits)
 *   "cholqr_passes"          as pfsm_set_cholqr_passes (1 | 2)
 * May allocate workspace (a newly selected route).  Errors: -1 handle, -2 unknown key, -3 value out of range,
 * 1000+cudaError.
 */
int pfsm_set_option(pfsm_handle_t h, const char* key, int64_t value);

/* Change alpha (it scales with 1/||A||^2, so it changes when the spectrum's extent does). */
int pfsm_set_alpha(pfsm_handle_t h, double alpha);

/* Bytes of device workspace the handle currently owns. */
size_t pfsm_workspace_bytes(pfsm_handle_t h);

/* Number of kernel launches (memsets and copies not counted) one pfsm_solve of this handle makes. */
int64_t pfsm_launches_per_solve(pfsm_handle_t h);

/*
 * Per-step device times of the NEXT solves: when enabled, pfsm_solve records CUDA events between the
 * steps; pfsm_get_step_ms synchronizes and returns ms for steps 2, 3, 4, 5 in ms[0..3].
 */
int pfsm_enable_step_timing(pfsm_handle_t h, int32_t enable);
int pfsm_get_step_ms(pfsm_handle_t h, float* ms4);

/*
 * Roofline calibration (no data, no memory traffic): runs a register-only loop of FP64 tensor
 * instructions (mma.sync m8n8k4 f64 -> SASS DMMA.8x8x4) on every SM and returns the issue-rate peak
 * in TFLOP/s measured with CUDA events.  kind 0 = DMMA, kind 1 = scalar DFMA.
 */
int pfsm_probe_fp64_peak(int32_t kind, void* stream, double* tflops);

/*
 * Step 5 WITHOUT ANY ALLOCATION, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid it): lambda_i = v_i^T A v_i and r_i = ||A v_i - lambda_i v_i||_2 (reading R11; the same two
 * kernels, operation order and bits as pfsm_rayleigh).  Needs no handle: the one piece of scratch, the N x N product
 * T = V A, lives in a static device array inside the library (8 MiB on every GPU that loads it, held until exit).
 *   N          matrix order: even, 2 <= N <= 1024; anything else returns PFSM_ERR_NOALLOC_SIZE
 *   A, V       device, N x N, leading dimension N, 16-byte aligned, read only (column i of V = vector i)
 *   lambda_out device, N (out)          resid_out  device, N (out)
 * Calls no cudaMalloc, cudaFree or allocating library routine; enqueues two kernels on `stream` and returns.
 * All calls on a device share the static array: it keeps the last call's contents (every call overwrites the part it reads,
 * nothing needs clearing), and two calls that overlap on the GPU -- different streams, no dependency -- RACE.  Serialize them.
 * Errors: PFSM_ERR_NOALLOC_SIZE, -2..-5 null or misaligned pointer, 1000+cudaError.
 */
#define PFSM_ERR_NOALLOC_SIZE 900
int pfsm_rayleigh_noalloc(int64_t N, const double* A, const double* V, double* lambda_out, double* resid_out, void* stream);

/* Static text for a return code of this API. */
const char* pfsm_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* PFSM_H */
