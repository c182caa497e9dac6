/*
 * bie.h -- C ABI of the B200-native boundary-integral hot path of arXiv 2108.01786
 *          (Ambrose, Camassa, Marzuola, McLaughlin, Robinson, Wilkening: "Numerical Algorithms for
 *          Water Waves with Background Flow over Obstacles and Topography").
 *
 * PAPER.md below is /root/reference/PAPER.md; a citation is a line range plus the equation it falls in.
 *
 * The path: (a) dense construction of the collocation matrix of Eq. (3.16) whose
 * entries are the periodised Cauchy kernel zeta'_j/2 cot((zeta_j - zeta_k)/2) of Table 1
 * on the trapezoidal rule, with the analytic diagonal limit
 * (PAPER.md:L265), the +-1/2 I of Eq. (3.10) and the rank-(N-1) stream-function
 * correction E_m; (b) restarted GMRES on that system: dense FP64
 * matvec, Gram-Schmidt, Givens rotations, all on the device.
 *
 * Conventions common to all calls
 *   - Everything is FP64.  Complex arrays are interleaved (re, im) doubles.
 *   - "dev" pointers are device memory of the ctx's GPU, caller-owned, 16-byte aligned; "host" pointers
 *     are ordinary host memory.  The library never frees or keeps caller buffers beyond a call, except
 *     that the node tables derived from the last geometry live in the ctx (O(n) bytes, grown on demand).
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Calls are
 *     asynchronous on it unless stated otherwise.
 *   - A ctx serves ONE stream at a time: its node tables, the matrix-free operator's tables and its staging
 *     buffers are shared by all calls, so calls on the same ctx must be issued on one stream, or be ordered by
 *     the caller (events) when the stream changes.  Use one ctx per concurrently used stream.  (The grid-barrier
 *     counter of a solve lives in that call's workspace, that of bie_matvec_free in a ring of counters, so an
 *     overlap of two launches cannot dead-lock the GPU; it can still give wrong numbers.)
 *   - The first matrix-free or hybrid call after a geometry change (bie_matvec_free, bie_gmres with A == NULL,
 *     bie_gmres_hybrid, bie_solve_host with those operators) builds the sparse matrix of near pairs and
 *     SYNCHRONISES the stream once to size it (the number of near pairs comes back to the host; no capacity limit).
 *   - Components: component 0 is the free surface Gamma_0, component 1 the bottom
 *     Gamma_1, components 2.. the obstacles, parameterised CLOCKWISE (fluid on the left of solids, on
 *     the right of Gamma_0).  counts[c] = M_c nodes at alpha_{cl} = 2 pi l / M_c;
 *     n = sum_c M_c.  Node arrays hold the components concatenated in this order.
 *   - Matrices are row-major, row = target node (k,m), column = source node (j,l), leading dimension
 *     lda >= n, lda even (so that every row is 16-byte aligned).
 *   - Return value: 0 = OK; > 0 = numerical status (BIE_MAX_ITERS: outputs still valid);
 *     < 0 = error, nothing useful was written.  -(100 + e) reports cudaError_t e.  No exceptions cross
 *     the ABI.  There is no CPU fallback: without an sm_100 device bie_create fails.
 */
#ifndef BIE_H
#define BIE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BIE_OK 0
#define BIE_MAX_ITERS 1        /* bie_gmres: max_iters reached before |g_{j+1}| <= tol ||b||        */
#define BIE_ERR_NULL (-1)      /* a required pointer is NULL                                        */
#define BIE_ERR_GEOMETRY (-2)  /* ncomp < 1, a count < 1, kinds not (0, 1?, 2, 2, ...), n too large  */
#define BIE_ERR_LAYOUT (-3)    /* lda < n, lda odd, or a device pointer not 16-byte aligned          */
#define BIE_ERR_WORKSPACE (-4) /* workspace too small (see bie_*_workspace_bytes)                    */
#define BIE_ERR_DEVICE (-5)    /* not a compute-capability-10.x device                               */
#define BIE_ERR_ARG (-6)       /* restart < 1, max_iters < 0, tol < 0, unknown variant/flags         */
#define BIE_ERR_NOALLOC_SIZE (-9) /* bie_gmres_noalloc: (n, restart) needs more than the static scratch */
#define BIE_ERR_CUDA_BASE (-100)

#define BIE_KIND_SURFACE 0
#define BIE_KIND_BOTTOM 1
#define BIE_KIND_OBSTACLE 2

/* operator of bie_solve_host (its `matrix_free` argument) */
#define BIE_OP_DENSE 0  /* whole matrix stored, GEMV from HBM                                            */
#define BIE_OP_FREE 1   /* nothing stored, entries recomputed on the fly                                 */
#define BIE_OP_HYBRID 2 /* leading block of bie_hybrid_cols(n) rows and columns stored, the rest recomputed */

/* bie_build `variant` */
#define BIE_VARIANT_A 0 /* Eq. (3.16): 1/2 I + K_mm - E_m on obstacle diagonal blocks  */
#define BIE_VARIANT_B 1 /* the uncorrected operator B of Eq. (3.10), for invariants    */
#define BIE_VARIANT_VORTEX 2 /* vortex-sheet system S of Eqs. (4.14) + (4.17), built from the
                                adjoint matrices of Eq. (4.7):  c+ = zeta'_k[m]/(2 M_j) cot((zeta_k[m] - zeta_j[l])/2)
                                  k = 0,  j = 0  :  Im c+ + 1/2 [s==t]     (1/2 I + K+_00)
                                  k = 0,  j >= 1 : -Re c+                  (-G+_j0)
                                  k >= 1, j = 0  :  Re c+                  (G+_0k)
                                  k >= 1, j >= 1 :  Im c+ - 1/2 [s==t]     (-1/2 I + K+_jk)
                                Its trailing block (rows and columns on solids: A + M_0 lda + M_0, size n - M_0, M_0 even)
                                is the auxiliary system (4.5); bie_gmres takes it as it is.
                                The matrix-free and hybrid operators also serve the full S (13 FP64 instructions per pair). */

typedef struct bie_ctx bie_ctx;

/* Creates a context on CUDA device `device` (makes it current for the calling thread during each call).
 * Fails with BIE_ERR_DEVICE unless the device has compute capability 10.x (B200: sm_100a code only). */
int bie_create(bie_ctx** ctx, int device);
int bie_destroy(bie_ctx* ctx);

/* Static, human-readable text for a return code. */
const char* bie_strerror(int code);

/* Number of SMs of the ctx's device and the FP64 FMA lanes per SM per clock the build roofline assumes
 * (64 on sm_100).  Used by bench.py for the "alu" roofline denominators. */
int bie_device_info(bie_ctx* ctx, int* sm_count, int* fp64_fma_per_sm_clk, int* l2_bytes_mib);

/* ---------------------------------------------------------------------------------------------------
 * (a) Matrix build, SURVEY 8(a) rows a1-a3.
 *
 * For target node t = (k,m) and source node s = (j,l), s != t (Table 1; weights
 * 1/M_j PAPER.md:L302):
 *        c = zeta'_j[l] / (2 M_j) * cot((zeta_j[l] - zeta_k[m]) / 2),
 * and for s == t the limit   c = zeta''_k[m] / (2 zeta'_k[m] M_k).   Entry A[t][s]:
 *        k = 0,  j = 0  :  Im c - 1/2 [s==t]                              (-1/2 I + K_00)
 *        k = 0,  j >= 1 :  Re c                                           (G_0j)
 *        k >= 1, j = 0  : -Re c                                           (-G_k0)
 *        k >= 1, j >= 1 :  Im c + 1/2 [s==t] - [k == j is an obstacle]/M_k   (1/2 I + K_kj - E_k)
 * (Eq. (3.10); Eq. (3.16) and E_m PAPER.md:L308-L324).  variant = BIE_VARIANT_B omits E_k.
 *
 * counts, kinds: host int32[ncomp].  kinds[0] must be BIE_KIND_SURFACE and no other component may be;
 * at most one BIE_KIND_BOTTOM.  zeta, dzeta, d2zeta: dev, interleaved complex, length n.  The values are
 * used exactly as given (no differentiation inside).  A: dev, n x lda doubles, fully overwritten in the
 * first n columns of its n rows.
 * Launches: one node-preparation kernel and one tile kernel.  The node tables stay in the ctx for
 * bie_matvec_free / bie_gmres(A == NULL).
 */
int bie_build(bie_ctx* ctx, int ncomp, const int32_t* counts, const int32_t* kinds,
              const double* zeta, const double* dzeta, const double* d2zeta,
              int variant, double* A, int64_t lda, void* stream);

/* rebuild only the blocks that involve component 0 (row block 0 and column block 0),
 * for a sequence of stages in which only the free surface moved (solids "do not change in time",
 * PAPER.md:L498).  Same arguments as bie_build; the solid-solid blocks of A are left untouched. */
int bie_build_update(bie_ctx* ctx, int ncomp, const int32_t* counts, const int32_t* kinds,
                     const double* zeta, const double* dzeta, const double* d2zeta,
                     int variant, double* A, int64_t lda, void* stream);

/* Hybrid operator (north_star: "matrix-free fused rebuild+matvec variant chosen by measurement").  The dense
 * GEMV is HBM-bound and leaves the FP64 pipe idle, the matrix-free operator is FP64-bound and leaves HBM idle;
 * the hybrid operator does both at once: the LEADING nblock x nblock block of the matrix is stored and arrives in
 * shared memory by bulk copies (TMA) while the warps of every CTA recompute every other entry from the node tables
 * -- with the symmetric pair loops (see bie_set_symmetric): every pair {t, s} outside the block has
 * max(t, s) >= nblock, so one evaluation of the pair serves both entries.
 * The block is kept in a BLOCK FORMAT private to the library: tiles of 4 rows x 512 columns, each tile contiguous
 * (16 KB, so that ONE bulk copy moves it), rows and columns padded to whole tiles; bie_hybrid_block_bytes(nblock)
 * is its size.  nblock must be a row-block boundary of the pair loops: a multiple of 128 up to M_0, or M_0 itself,
 * or M_0 plus a multiple of 128; even; < n.
 * bie_build_block: the entries of bie_build for rows and columns [0, nblock), written in the block format to A
 *   (dev, bie_hybrid_block_bytes(nblock) bytes, 16-byte aligned).
 * bie_build_cols: as bie_build (row-major), but only the columns [0, ncols) of every row are written (1 <= ncols <= n).
 * bie_hybrid_cols: the block edge the library recommends for n on a B200 (0 = too small, use bie_gmres); it uses M_0
 *   of the ctx's current geometry when that has n nodes, else assumes M_0 is a multiple of 128.
 * bie_set_hybrid_free_warps: tuning knob, warps per CTA on the pair loops (1..15; default 12 = the warps of three of the
 *   SM's four sub-partitions, the fourth hosts the warp that issues the bulk copies and three warps that multiply the
 *   landed tiles; other values: warps 0..w-1 run the pair loops, the others up to 14 consume tiles, 15 issues). */
size_t bie_hybrid_block_bytes(int nblock);
int bie_build_block(bie_ctx* ctx, int ncomp, const int32_t* counts, const int32_t* kinds,
                    const double* zeta, const double* dzeta, const double* d2zeta,
                    int variant, int nblock, double* A, void* stream);
int bie_build_cols(bie_ctx* ctx, int ncomp, const int32_t* counts, const int32_t* kinds,
                   const double* zeta, const double* dzeta, const double* d2zeta,
                   int variant, int ncols, double* A, int64_t lda, void* stream);
int bie_hybrid_cols(bie_ctx* ctx, int n);
int bie_set_hybrid_free_warps(bie_ctx* ctx, int free_warps);
/* tuning knob: tiles of the stored block a pair-loop warp may take between two of its source chunks (0..64; 0: only the
 * warps above bie_set_hybrid_free_warps consume the block) */
int bie_set_hybrid_poll_tiles(bie_ctx* ctx, int tiles);

/* Prepares the node tables of a geometry in the ctx without writing a matrix (for the matrix-free
 * operator).  Same geometry arguments as bie_build. */
int bie_set_geometry(bie_ctx* ctx, int ncomp, const int32_t* counts, const int32_t* kinds,
                     const double* zeta, const double* dzeta, const double* d2zeta,
                     int variant, void* stream);

/* ---------------------------------------------------------------------------------------------------
 * (b) Matvec:  y = A x   (dev, dev, dev; x and y of length n, must not alias).
 * bie_matvec reads the stored matrix (HBM-bound); bie_matvec_free recomputes the entries of the geometry
 * last given to bie_build / bie_set_geometry on the fly (FP64-bound, no matrix traffic).
 */
int bie_matvec(bie_ctx* ctx, int n, const double* A, int64_t lda, const double* x, double* y, void* stream);
int bie_matvec_free(bie_ctx* ctx, int n, const double* x, double* y, void* stream);
/* The matrix-free operator (bie_matvec_free, bie_gmres with A == NULL) and the recomputed part of the hybrid operator
 * (variants A and B, n <= 65536) use the oddness of the kernel, cot((zeta_s - zeta_t)/2) = -cot((zeta_t - zeta_s)/2): one
 * evaluation of the pair serves the entries (t,s) and (s,t) (13 FP64 instructions for two entries instead of 20).
 * on = 0 switches to the one-directional pair loops, on = 1 (default; 2 is accepted as a synonym) uses the symmetric
 * ones.  Same results to rounding; all are deterministic. */
int bie_set_symmetric(bie_ctx* ctx, int on);

/* Small stored-matrix solves (n <= 640 at restart 50): bie_gmres and bie_gmres_noalloc run the same restarted GMRES (rows a5-a10;
 * PAPER.md:L855, stopping rule PAPER.md:L869) on ONE thread-block cluster of 16 (else 8) CTAs -- the rows of A and of the
 * Krylov basis in the CTAs' shared memory, exchanges by asynchronous stores into the peers' shared memory with mbarrier
 * transaction counts instead of grid barriers and L2 round trips -- when all but four rows of A per CTA fit and the device can
 * co-schedule such a cluster; otherwise, and for larger n, the grid-wide kernel.  Same arguments, workspace, outputs and
 * tolerances; deterministic; iteration counts of the two kernels agree within one step (their sums differ in order).
 * on = 1 (default) / 0: use it / never use it. */
int bie_set_small_gmres(bie_ctx* ctx, int on);

/* stream function prescribed on the solids, circulation parameters
 * a_m = <1_m, omega> unknown.  Adds, in place, the rank-(N-1) correction of Eq. (B.2) to a matrix A that holds
 * the operator B (bie_build with BIE_VARIANT_B):  A[t][s] += c_m[t]/M_m for every column s of obstacle m, with
 * c_m[t] = phi_cyl(zeta_t - z_m) = arg(1 - e^{i(zeta_t - z_m)}) for rows on Gamma_0 and psi_cyl = -log|1 - e^{i(zeta_t - z_m)}|
 * for rows on solids (Phi_cyl = -i log(1 - e^{iz}), Eq. (3.2)).  centers: HOST, interleaved (re, im), one
 * point z_m inside each obstacle, in component order; zeta: dev as in bie_build; A: dev, n x lda.
 * The right-hand side of the variant is b_0 = phi - V_1 xi, b_k = psi|_k - V_1 eta_k; solve with bie_gmres. */
int bie_add_cyl_columns(bie_ctx* ctx, int ncomp, const int32_t* counts, const int32_t* kinds, const double* zeta,
                        const double* centers, double* A, int64_t lda, void* stream);

/* values in the closed fluid region of nf
 * (1..4) functions analytic in the fluid, from their boundary values, spectrally accurate up to the boundary:
 *      f(z) = sum_s lambda~_s(z) f_s / sum_s lambda~_s(z),   lambda~_s(z) = (sigma_k/M_k) 1/2 cot((zeta_s - z)/2) zeta'_s     (Eq. F.4 / 5.5)
 * with sigma_0 = -1 on Gamma_0 (parameterised with the fluid on its right) and +1 on the solids; a point that
 * coincides with a node (modulo the period) gets that node's value.  E.g. f = Phi' and Phi_t for the velocity
 * and pressure fields of Eq. (5.3)-(5.4).  zeta, dzeta: dev, as in bie_build (d2zeta is not needed); fvals: dev, [nf][n] complex
 * interleaved; zpts: dev, npts complex; out: dev, [nf][npts] complex; workspace: dev, bie_cauchy_eval_workspace_bytes(). */
size_t bie_cauchy_eval_workspace_bytes(bie_ctx* ctx, int nf, int npts);
int bie_cauchy_eval(bie_ctx* ctx, int ncomp, const int32_t* counts, const int32_t* kinds,
                    const double* zeta, const double* dzeta, int nf, const double* fvals,
                    int npts, const double* zpts, double* out, void* workspace, size_t workspace_bytes, void* stream);

/* y (nrows) = A (nrows x ncols, row-major, lda >= ncols even) x (ncols): the same HBM-bound kernel on a rectangular block. */
int bie_matvec_rect(bie_ctx* ctx, int nrows, int ncols, const double* A, int64_t lda, const double* x, double* y,
                    void* stream);

/* ---------------------------------------------------------------------------------------------------
 * (b') Normal velocity on the free surface after the solve, Section 3.4, SURVEY 8(f) NEXT-2.
 * Writes the M_0 x n matrix Nmat (row-major, lda >= n even) with
 *      s_alpha d phi~/dn (alpha_m) = sum_s Nmat[m][s] omega'[s]
 *                                  = -1/2 H omega'_0 - G+_00 omega'_0 + sum_{j>=1} K+_j0 omega'_j     (Eqs. 3.24 + 3.19),
 * omega' = the derivatives of the densities (all components concatenated; the caller differentiates, e.g. by FFT).
 * Row m on Gamma_0, column (j,l):  c+ = zeta'_0[m]/(2 M_j) cot((zeta_0[m] - zeta_j[l])/2)   (integration variable in
 * the first slot of the kernels):
 *      j >= 1 :  Im c+                                                         (K_j0(alpha_jl, alpha_m)/M_j)
 *      j = 0  : -Re c+ + kappa_{m-l},  diagonal -Re{zeta''_0/(2 zeta'_0)}/M_0   (-G_00(alpha_l, alpha_m)/M_0 - 1/2 H)
 * where kappa_d carries the regulariser 1/2 cot((alpha - beta)/2) of G_00 (Table 1) and -1/2 of the
 * Hilbert transform of Eq. (3.22) in its exact discrete form (symbol -i sgn k, Nyquist mode dropped):
 *      kappa_d = (-1)^d cot(pi d/M_0)/(2 M_0)  (M_0 even),   (-1)^d/(2 M_0 sin(pi d/M_0))  (M_0 odd),   kappa_0 = 0.
 * The phi_mv term (3.17) is pointwise input data and is not included.  Apply with bie_matvec_rect(M_0, n, ...).
 * The call replaces the ctx's node tables (call bie_set_geometry / bie_build again before a matrix-free solve). */
int bie_build_normal_velocity(bie_ctx* ctx, int ncomp, const int32_t* counts, const int32_t* kinds,
                              const double* zeta, const double* dzeta, const double* d2zeta,
                              double* Nmat, int64_t lda, void* stream);

/* ---------------------------------------------------------------------------------------------------
 * (c) Restarted GMRES(restart), SURVEY 8(a) rows a5-a10 (Saad & Schultz, ref. [38] cited at
 * PAPER.md:L855), unpreconditioned, x0 = 0, on the system as stored:
 *   cycle:  r = b - A x (first cycle r = b), beta = ||r||, v_1 = r/beta, g = beta e_1;
 *   step j: w = A v_j; orthogonalise w against v_1..v_j by classical Gram-Schmidt applied twice (CGS2);
 *           h_{j+1,j} = ||w||, v_{j+1} = w/h_{j+1,j}; previous Givens rotations on column j of H, new
 *           rotation, g_{j+1} = -s_j g_j; iters += 1; stop when |g_{j+1}| <= tol * ||b||
 *           (the criterion behind i_max) or iters == max_iters;
 *   cycle end: y = R^{-1} g, x += V y; restart if not converged.
 * The whole solve is ONE cooperative kernel launch; nothing returns to the host until it ends.
 *
 * A == NULL selects the matrix-free operator of the ctx's current geometry (then lda is ignored and n must
 * match it).  rhs, x: dev, length n.  iters_out (int32) and relres_out (double: TRUE relative residual
 * ||b - A x|| / ||b||, reported, never used to continue) are DEVICE pointers (may be NULL).
 * workspace: dev, at least bie_gmres_workspace_bytes(n, restart) bytes, contents undefined afterwards.
 * Returns BIE_OK immediately after the launch (convergence status is in *iters_out vs max_iters, and in
 * status_out if not NULL: dev int32, 0 converged / 1 max_iters / 2 breakdown (h_{j+1,j} == 0, converged)).
 * res_hist (dev, max_iters + 1 doubles, may be NULL): res_hist[i] = recurrence residual |g_{i+1}| / ||b|| after
 * i steps (res_hist[0] = 1), the quantity behind the paper's i_max statistics.
 */
size_t bie_gmres_workspace_bytes(int n, int restart);
int bie_gmres(bie_ctx* ctx, int n, const double* A, int64_t lda, const double* rhs,
              double tol, int restart, int max_iters,
              double* x, int32_t* iters_out, double* relres_out, int32_t* status_out, double* res_hist,
              void* workspace, size_t workspace_bytes, void* stream);

/* The same solve with the stored matrix for callers that must not allocate (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): there is no workspace argument, the workspace is a file-scope device
 * array of BIE_NOALLOC_SCRATCH_BYTES inside the library (every GPU that loads the library holds it until exit), and the
 * call itself calls no cudaMalloc, cudaFree or allocating library routine.  The ctx must exist already (bie_create
 * allocates; do that at set-up).  The first call on a device looks up the array's device address (cudaGetSymbolAddress,
 * not an allocation).
 * A != NULL (dev, lda as in bie_gmres): only the stored-matrix operator is served -- the matrix-free and hybrid operators
 * build a near matrix whose size depends on the geometry.  rhs, x, iters_out, relres_out, status_out: as in bie_gmres.
 * Limit: bie_gmres_workspace_bytes(n, restart) <= BIE_NOALLOC_SCRATCH_BYTES (4 MiB: n = 4608 with restart 50 takes
 * 2.3 MB, n = 8192 with restart 50 3.8 MB); anything larger returns BIE_ERR_NOALLOC_SIZE and launches nothing.
 * ALL calls, from all ctxs and streams of a process, share the one array per device: two calls that overlap on the GPU
 * race (keep them on one stream or order them with events).  The array keeps the previous call's contents; the solve
 * writes every part before reading it and clears the grid-barrier counter on the stream before the launch. */
#define BIE_NOALLOC_SCRATCH_BYTES (4u << 20)
size_t bie_gmres_noalloc_max_bytes(void);
int bie_gmres_noalloc(bie_ctx* ctx, int n, const double* A, int64_t lda, const double* rhs,
                      double tol, int restart, int max_iters,
                      double* x, int32_t* iters_out, double* relres_out, int32_t* status_out, void* stream);

/* Same solve with the hybrid operator: A holds the leading ncols_dense x ncols_dense block of the matrix of the ctx's
 * current geometry in the block format (bie_build_block), ncols_dense a row-block boundary as described at
 * bie_build_block (else BIE_ERR_ARG).  Everything else as bie_gmres. */
int bie_gmres_hybrid(bie_ctx* ctx, int n, const double* A, int ncols_dense, const double* rhs,
                     double tol, int restart, int max_iters,
                     double* x, int32_t* iters_out, double* relres_out, int32_t* status_out, double* res_hist,
                     void* workspace, size_t workspace_bytes, void* stream);

/* ---------------------------------------------------------------------------------------------------
 * End-to-end call with HOST buffers (what bench.py's "e2e" times): copies the node data and rhs to the
 * device, builds A, solves, copies x / iters / relres back and SYNCHRONISES the stream before returning.
 * zeta, dzeta, d2zeta, rhs, x: host (pinned memory makes the copies asynchronous).  dev_workspace: dev, at
 * least bie_solve_workspace_bytes(n, restart) bytes (holds node data, A with lda = n rounded up to even,
 * rhs, x and the GMRES workspace).  matrix_free selects the operator: BIE_OP_DENSE (0), BIE_OP_FREE (1: no
 * matrix is stored) or BIE_OP_HYBRID (2: the leading block of bie_hybrid_cols(n) rows and columns is stored; falls
 * back to BIE_OP_FREE when n is too small for a block).  Returns BIE_OK,
 * BIE_MAX_ITERS or an error.
 */
size_t bie_solve_workspace_bytes(int n, int restart, int matrix_free);
int bie_solve_host(bie_ctx* ctx, int ncomp, const int32_t* counts, const int32_t* kinds,
                   const double* zeta, const double* dzeta, const double* d2zeta, const double* rhs,
                   double tol, int restart, int max_iters, int matrix_free,
                   double* x, int32_t* iters_out, double* relres_out,
                   void* dev_workspace, size_t dev_workspace_bytes, void* stream);

/* ---------------------------------------------------------------------------------------------------
 * Roofline probe (measurement support, not part of the method): launches a kernel of dependent-chain-free
 * DFMA work, `fma_per_thread` FMAs in each of grid*block threads filling every SM, so that bench.py can
 * time the FP64 pipe's sustained rate on this very GPU.  out: dev, >= 8 bytes (keeps the work alive).
 * *total_fma (host) receives the number of FMAs issued.
 */
int bie_probe_dfma(bie_ctx* ctx, int64_t fma_per_thread, double* out, int64_t* total_fma, void* stream);
/* Read-only streaming probe: sums nbytes (multiple of 16) of `buf` (dev, 16-byte aligned) with 128-bit evict-first loads
 * from every SM, the access pattern of the GEMV, so that bench.py can quote the GEMV against a READ peak measured in the
 * same run (MEASURED_PEAKS.json's number is a read+write copy).  out: dev, >= 8 bytes. */
int bie_probe_read(bie_ctx* ctx, const double* buf, int64_t nbytes, double* out, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* BIE_H */
