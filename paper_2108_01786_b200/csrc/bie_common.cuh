// bie_common.cuh -- shared declarations of the CUDA path (sm_100a only).  No oracle code is shared.
//
// Pair arithmetic (DESIGN.md section 5 "Pair arithmetic").  The periodised Cauchy kernel of Eq. (3.4)
// for a source node s and a target node t, w = zeta_s - zeta_t, is evaluated from ONE complex
// exponential per NODE, E = e^{i zeta} = e^{-(y - y_ref)} (cos x + i sin x), M = |E|^2, with no transcendental
// per pair:
//     cot(w/2) = i (e^{iw} + 1)/(e^{iw} - 1) = i (E_s + E_t) conj(E_s - E_t) / |E_s - E_t|^2
//              = ( -2 X + i Y ) / den,    X = Im(E_t conj E_s),  Y = M_s - M_t,  den = |E_s - E_t|^2 .
// With the source weight q_s = zeta'_s/(2 M_j) the entry is (alpha X + beta Y)/den:
//     Im{q cot} : (alpha, beta) = (-2 qi,  qr)     Re{q cot} : (-2 qr, -qi)     -Re{q cot} : (2 qr, qi)
// "Difference form" (Eq. (3.16) build and its matrix-free operator): with d = E_s - E_t = dr + i di, which den
// needs anyway,  X = Ei_s dr - Er_s di  and  Y = 2 (Er_s dr + Ei_s di) - den,  so that
//     (alpha X + beta Y)/den = (U_s dr + W_s di)/den - beta,   U_s = alpha Ei_s + 2 beta Er_s,  W_s = 2 beta Ei_s - alpha Er_s:
// the numerator costs 2 FP64 instructions from per-SOURCE constants and the constant -beta (the far-field limit
// cot -> -+i) is added per entry by the final FMA of the build (10 FP64-pipe instructions per entry: 2 sub, 2 den,
// 2 numerator, 3 reciprocal (bie_rcp3), 1 FMA) or, in the matrix-free operator, once per application as
// -sum_s beta_s x_s (10 per pair including the accumulation).  The vortex-sheet / normal-velocity builds, whose weight
// belongs to the ROW node, keep the (X, Y) form (13 per entry).  E_s - E_t cancels for |w| -> 0 (relative error of d
// about eps/|w|, entry error a few eps |q_s|/|w|^2); pairs with den < thr_s = tau_s M_s, tau_s = BIE_NEAR_C |q_s|
// (clamped), are "near": they are recomputed from the coordinate differences with the Laurent series of cot
// (bie_cot_half_near), accurate to rounding, and the pair s == t takes the analytic diagonal limit.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/bie.h"

#define BIE_MAX_COMP 64
#define BIE_VARIANT_NORMAL_INTERNAL 3  // node tables for bie_build_normal_velocity (not a bie_build variant)
#define BIE_NODE_PAD 256              // node tables are padded to a multiple of the build tile width
#define BIE_NEAR_C 0.25               // tau_s = BIE_NEAR_C |q_s|  (fast-path entry error <= ~1e-14)
#define BIE_NEAR_TAU_MIN 1.0e-9
#define BIE_NEAR_TAU_MAX 1.0e-2       // |w| < 0.1: Laurent truncation 2|w/2|^9/93555 < 1e-16
#define BIE_HYBRID_POLL_TILES 0         // hybrid operator: tiles of the stored block a pair-loop warp may take between two source chunks
#define BIE_HYBRID_FREE_WARPS 12       // hybrid operator: warps of a CTA on the pair loops (of 16; one warp issues the bulk copies)
#define BIE_HYBRID_DENSE_FRACTION 0.5625 // hybrid operator: edge of the stored leading block as a share of n (32 % of the entries)
#define BIE_CLUSTER_MAX_N 1024         // stored-matrix GMRES on one thread-block cluster at most up to this n (bie_gmres_cluster.cu)
#define BIE_CLUSTER_NOT_TAKEN 1        // bie_launch_gmres_cluster: not for the cluster kernel, use the grid-wide one
#define BIE_SYNC_SLOTS 16             // grid-barrier counters of a ctx (bie_matvec_free cycles through them), 256 B apart

// Node table, arrays of double2 of length npad.
struct NodeTable {
    const double2* E;    // (Re, Im) of e^{i zeta} scaled by e^{y_ref}
    const double2* MT;   // (M = |E|^2, thr = tau_s M)
    const double2* Q;    // zeta' / (2 M_j)   (source weight)
    const double2* XY;   // (Re zeta, Im zeta)  (near path)
    const double2* DG;   // (complete diagonal entry Im{zeta''/(2 zeta')}/M_k -+ 1/2 - em,  em = [obstacle, variant A]/M_k)
    const int* COMP;     // component index of the node (padding: -1)
    int n;
    int npad;
};
#define BIE_NODE_ARRAYS 10            // doubles per node in node_buf

// component offsets, by value into kernels (<= 260 bytes)
struct CompTable {
    int ncomp;
    int off[BIE_MAX_COMP + 1];
};

struct bie_ctx {
    int device;
    int sm_count;
    int l2_bytes;
    int coop_ok;
    int max_smem_optin;
    // node-table storage (device), capacity in nodes
    double* node_buf;
    int* comp_buf;
    double* free_buf;        // matrix-free operator: per-matvec source tables [8][cap] + partial sums (bie_free.cuh)
    double* taubar;          // device scalar: max_s tau_s of the current geometry (bie_near.cu)
    int* near_ptr;           // CSR near matrix (bie_near.cu): [8 cap + 1] offsets of the (row, segment) lists
    int* near_col;           // [near_cap] column indices, grown to the scanned total (bie_ensure_near)
    double* near_val;        // [near_cap]
    size_t near_cap;         // entries allocated in near_col / near_val
    int near_valid;          // near matrix built for the current geometry
    double* pc_buf;          // symmetric matrix-free operator: reverse partials [row blocks][npad] (bie_free_sym.cuh)
    size_t pc_cap;           // doubles allocated in pc_buf
    char* sym_tab;           // device tables of the symmetric work list (cum, perm, pos), cached per geometry and split
    size_t sym_tab_bytes;
    long long sym_key[4];    // (geometry generation, s_off, grid, 1) the cached tables were made for
    long long sym_U;         // their total number of list positions
    long long geom_gen;      // incremented by every bie_prepare_nodes
    int smem_set[16];        // dynamic shared memory already granted to the kernel instantiations (cudaFuncSetAttribute once)
    int use_sym;             // use the symmetric work split for the whole-matrix matrix-free operator
    double* kappa;           // [cap] real-cot table of the normal-velocity operator (bie_build_normal_velocity)
    int hybrid_free_warps;   // hybrid operator: warps per CTA on the pair loops (warps above it only consume tiles; warp 15 issues the copies)
    int hybrid_poll_tiles;   // hybrid operator: tiles a pair-loop warp may take between two source chunks (0: it never does)
    unsigned int* sync_buf;  // BIE_SYNC_SLOTS grid-barrier counters (256 B apart) + two device scalars behind them
    int sync_next;           // next counter slot (bie_matvec_free); bie_gmres keeps its counter in the caller's workspace
    int small_gmres;         // bie_set_small_gmres: small stored-matrix solves run on one thread-block cluster (default 1)
    int cluster_size;        // 0: not probed yet; -1: the device cannot co-schedule such a cluster; else 16 or 8
    int cap;
    // current geometry (host copies)
    int have_geom;
    int n;
    int ncomp;
    int variant;
    int counts[BIE_MAX_COMP];
    int kinds[BIE_MAX_COMP];
    CompTable comps;
    // staging for bie_solve_host
    int32_t* pinned_i;  // [4]
    double* pinned_d;   // [4]
};

static inline int bie_cuda_err(cudaError_t e) { return e == cudaSuccess ? BIE_OK : BIE_ERR_CUDA_BASE - (int)e; }
#define BIE_CUDA(call)                                    \
    do {                                                  \
        cudaError_t e__ = (call);                         \
        if (e__ != cudaSuccess) return bie_cuda_err(e__); \
    } while (0)

// row pairs per CTA block that a streaming GEMV keeps L2-resident (bie_gemv.cuh): about 60 % of the L2 (measured flat from
// 30 % to 60 %, worse above), less the bytes the caller keeps there anyway (Krylov basis), spread over the CTAs' row blocks
static inline int bie_gemv_resident_pairs(int l2_bytes, int nrows, long long lda, int rows_per_cta, size_t other_bytes)
{
    const double budget = 0.6 * (double)l2_bytes - (double)other_bytes;
    if (budget <= 0.0 || nrows < 1) return 0;
    const double frac = budget / ((double)nrows * (double)lda * 8.0);
    if (frac >= 1.0) return (rows_per_cta + 1) / 2;
    return (int)(frac * rows_per_cta) / 2;
}

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) once per kernel instantiation (slot) and ctx, again only when a call
// needs more than was granted before
template <typename K>
static inline int bie_grant_smem(bie_ctx* ctx, int slot, K kernel, size_t smem)
{
    if ((int)smem > ctx->smem_set[slot]) {
        BIE_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        ctx->smem_set[slot] = (int)smem;
    }
    return BIE_OK;
}

// Block format of the hybrid operator's stored leading block (bie_build_block -> bie_gmres_hybrid): tiles of
// BIE_TILE_ROWS rows x BIE_TILE_COLS columns, each tile contiguous (16 KB, row-major inside), tiles in row-major order of
// (row group, column chunk); rows and columns are padded to whole tiles (the padding is never read).  One tile = ONE
// bulk copy into shared memory: the TMA engine needs copies of this size to reach HBM speed (4 KB copies: 3.9 TB/s).
#define BIE_TILE_ROWS 4
#define BIE_TILE_COLS 512
static inline size_t bie_block_doubles(int nblock)
{
    const size_t ngrp = ((size_t)nblock + BIE_TILE_ROWS - 1) / BIE_TILE_ROWS, nch = ((size_t)nblock + BIE_TILE_COLS - 1) / BIE_TILE_COLS;
    return ngrp * nch * (BIE_TILE_ROWS * BIE_TILE_COLS);
}
#ifdef __CUDACC__
// offset of entry (t, s): row-major with leading dimension lda, or (lda == 0) the block format with nchT column chunks
__device__ __forceinline__ long long bie_entry_off(long long lda, int nchT, int t, int s)
{
    if (lda) return (long long)t * lda + s;
    return ((long long)(t / BIE_TILE_ROWS) * nchT + (s / BIE_TILE_COLS)) * (BIE_TILE_ROWS * BIE_TILE_COLS) +
           (long long)((t % BIE_TILE_ROWS) * BIE_TILE_COLS + (s % BIE_TILE_COLS));
}
#endif

static inline int bie_npad(int n) { return (n + BIE_NODE_PAD - 1) / BIE_NODE_PAD * BIE_NODE_PAD; }
// do the pair loops of the current geometry use the symmetric split (bie_free_sym.cuh)?  Eq. (3.16) variants, and while the
// reverse partials [row blocks][npad] stay small.  The near matrix is built for one or the other (bie_near.cu).
static inline bool bie_uses_sym(const bie_ctx* ctx)
{
    return ctx->use_sym != 0 && ctx->variant != BIE_VARIANT_VORTEX && bie_npad(ctx->n) <= 65536;
}
NodeTable bie_node_table(const bie_ctx* ctx);
struct FreePlan;
// doubles of ctx->free_buf for a node capacity `cap`; work split of the matrix-free operator over `grid` CTAs
size_t bie_free_buf_doubles(int cap);
int bie_free_plan(bie_ctx* ctx, int grid, int s_off, FreePlan* fp, cudaStream_t st);
int bie_ensure_near(bie_ctx* ctx, cudaStream_t st);

// internal entry points (one per .cu)
int bie_prepare_nodes(bie_ctx* ctx, int ncomp, const int32_t* counts, const int32_t* kinds,
                      const double* zeta, const double* dzeta, const double* d2zeta, int variant,
                      cudaStream_t st);
int bie_launch_build(bie_ctx* ctx, double* A, int64_t lda, int ncols, int nrows, int only_comp0, cudaStream_t st);
int bie_launch_matvec(bie_ctx* ctx, int nrows, int n, const double* A, int64_t lda, const double* x, double* y,
                      cudaStream_t st);
int bie_launch_matvec_free(bie_ctx* ctx, const double* x, double* y, cudaStream_t st);
// bie_gmres_cluster.cu: BIE_OK when the solve was launched on one thread-block cluster, BIE_CLUSTER_NOT_TAKEN when it is not for it
int bie_launch_gmres_cluster(bie_ctx* ctx, int n, const double* A, int64_t lda, const double* rhs, double tol, int restart,
                             int max_iters, double* x, int32_t* iters_out, double* relres_out, int32_t* status_out,
                             double* res_hist, double* Vg, int nld, double* R, cudaStream_t st);
int bie_launch_gmres(bie_ctx* ctx, int n, const double* A, int64_t lda, int nd, const double* rhs, double tol,
                     int restart, int max_iters, double* x, int32_t* iters_out, double* relres_out,
                     int32_t* status_out, double* res_hist, void* ws, size_t ws_bytes, cudaStream_t st);
size_t bie_gmres_ws_bytes(int n, int restart);
size_t bie_cauchy_eval_ws_bytes(int nf, int npts, int sm_count);
int bie_launch_cauchy_eval(bie_ctx* ctx, int ncomp, const int32_t* counts, const int32_t* kinds, const double* zeta,
                           const double* dzeta, int nf, const double* fvals, int npts, const double* zpts, double* out,
                           void* ws, size_t ws_bytes, cudaStream_t st);
int bie_launch_add_cyl_columns(bie_ctx* ctx, int ncomp, const int32_t* counts, const int32_t* kinds, const double* zeta,
                               const double* centers, double* A, int64_t lda, cudaStream_t st);
int bie_launch_probe_dfma(bie_ctx* ctx, int64_t fma_per_thread, double* out, int64_t* total_fma, cudaStream_t st);

// ---------------------------------------------------------------------------------------------------
// device helpers
// ---------------------------------------------------------------------------------------------------
#ifdef __CUDACC__
// 1/d for d > 0 in normal range: MUFU.RCP64H seed (relative error < 2^-19.9, measured over 2^24 arguments on
// B200) + one cubic refinement r0 (1 + e + e^2), e = 1 - d r0: error e^3 < 2^-59 plus rounding, 2 ulp at most.
// Three DFMA, no IEEE division sequence, no slow-path branch.  d = 0 gives inf/NaN: those pairs are near pairs
// and never use the value.
__device__ __forceinline__ double bie_rcp3(double d) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
    const double e = fma(-d, r, 1.0);
    const double t = fma(e, e, e);
    return fma(r, t, r);
}

// Near path: cot(w/2) for |w mod 2 pi| < 0.1, from the differences x = x_s - x_t, y = y_s - y_t.
// x is reduced to (-pi, pi] with a two-word 2 pi (the kernel is 2 pi-periodic in x: the sum over images
// of Eq. (3.4)), then with z = w/2
//   cot z = 1/z - z (1/3 + z^2 (1/45 + z^2 (2/945 + z^2/4725)))      (truncation < 1e-20 |z| for |z| < 0.03)
__device__ __forceinline__ void bie_cot_half_near(double x, double y, double* re, double* im) {
    const double TWO_PI_HI = 6.283185307179586232e+00, TWO_PI_LO = 2.449293598294706414e-16;
    const double k = rint(x * 0.15915494309189534561);
    x = fma(-k, TWO_PI_HI, x);
    x = fma(-k, TWO_PI_LO, x);
    const double zr = 0.5 * x, zi = 0.5 * y;
    const double m2 = fma(zr, zr, zi * zi);
    const double inv = 1.0 / m2;
    const double z2r = fma(zr, zr, -zi * zi), z2i = 2.0 * zr * zi;
    // Horner in z^2 (complex)
    double pr = 1.0 / 4725.0, pi = 0.0, tr;
    tr = fma(pr, z2r, -pi * z2i) + 2.0 / 945.0; pi = fma(pr, z2i, pi * z2r); pr = tr;
    tr = fma(pr, z2r, -pi * z2i) + 1.0 / 45.0;  pi = fma(pr, z2i, pi * z2r); pr = tr;
    tr = fma(pr, z2r, -pi * z2i) + 1.0 / 3.0;   pi = fma(pr, z2i, pi * z2r); pr = tr;
    // 1/z - z p
    *re = zr * inv - fma(zr, pr, -zi * pi);
    *im = -zi * inv - fma(zr, pi, zi * pr);
}

#ifndef BIE_BARRIER_RELACQ
#define BIE_BARRIER_RELACQ 1
#endif
// ---- grid barrier (cooperative launch guarantees co-residency) -------------------------------------
__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int* p)
{
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void grid_barrier(unsigned int* ctr, unsigned int& target)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        target += gridDim.x;
#if BIE_BARRIER_RELACQ
        // release on the arrival (cumulative over the writes the CTA's threads made before the block barrier above), acquire on
        // the poll: no separate fences
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" :: "l"(ctr) : "memory");
        while (ld_acquire_u32(ctr) < target) { }
#else
        __threadfence();
        atomicAdd(ctr, 1u);
        while (ld_acquire_u32(ctr) < target) { }
        __threadfence();
#endif
    }
    __syncthreads();
}

// a team = a contiguous group of warps of one CTA with its own named barrier (the whole CTA: barrier 0)
struct Team {
    int tid, nthr;     // thread index within the team, threads of the team (multiple of 32)
    int warp, nwarp;   // warp index within the team, warps of the team
    int bar;           // named barrier id
};
__device__ __forceinline__ void team_sync(const Team& t)
{
    asm volatile("bar.sync %0, %1;" ::"r"(t.bar), "r"(t.nthr) : "memory");
}
__device__ __forceinline__ Team cta_team()
{
    Team t;
    t.tid = threadIdx.x; t.nthr = blockDim.x; t.warp = threadIdx.x >> 5; t.nwarp = blockDim.x >> 5; t.bar = 0;
    return t;
}
// warps [w0, w0 + nw) of the CTA as a team using barrier `bar` (1..15); call only from those warps
__device__ __forceinline__ Team sub_team(int w0, int nw, int bar)
{
    Team t;
    t.tid = threadIdx.x - 32 * w0; t.nthr = 32 * nw; t.warp = (threadIdx.x >> 5) - w0; t.nwarp = nw; t.bar = bar;
    return t;
}

__device__ __forceinline__ double bie_warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
#endif
