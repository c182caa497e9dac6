// bie_api.cu -- the extern "C" boundary declared in include/bie.h: argument checks, ctx life cycle, the
// host-buffer end-to-end call and the DFMA roofline probe.  All arithmetic of the method is in the kernels
// of bie_nodes.cu / bie_build.cu / bie_matvec.cu / bie_gmres.cu.
#include <cstdlib>
#include <new>
#include "bie_common.cuh"

extern "C" {

int bie_create(bie_ctx** out, int device)
{
    if (!out) return BIE_ERR_NULL;
    *out = nullptr;
    int count = 0;
    cudaError_t e = cudaGetDeviceCount(&count);
    if (e != cudaSuccess || device < 0 || device >= count) return BIE_ERR_DEVICE;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return BIE_ERR_DEVICE;
    if (prop.major != 10) return BIE_ERR_DEVICE;  // sm_100a code only; there is no fallback path
    BIE_CUDA(cudaSetDevice(device));
    bie_ctx* c = new (std::nothrow) bie_ctx();
    if (!c) return BIE_ERR_CUDA_BASE - (int)cudaErrorMemoryAllocation;
    c->device = device;
    c->sm_count = prop.multiProcessorCount;
    c->l2_bytes = prop.l2CacheSize;
    c->coop_ok = prop.cooperativeLaunch;
    c->max_smem_optin = (int)prop.sharedMemPerBlockOptin;
    c->node_buf = nullptr; c->comp_buf = nullptr; c->free_buf = nullptr; c->cap = 0; c->have_geom = 0; c->n = 0;
    c->sync_buf = nullptr; c->pinned_i = nullptr; c->pinned_d = nullptr;
    c->near_ptr = nullptr; c->near_col = nullptr; c->near_val = nullptr; c->near_valid = 0; c->near_cap = 0;
    c->hybrid_free_warps = BIE_HYBRID_FREE_WARPS;
    c->hybrid_poll_tiles = BIE_HYBRID_POLL_TILES;
    c->taubar = nullptr; c->kappa = nullptr;
    c->pc_buf = nullptr; c->pc_cap = 0;
    c->sym_tab = nullptr; c->sym_tab_bytes = 0; c->sym_U = 0; c->geom_gen = 0; c->sync_next = 0;
    for (int i = 0; i < 4; ++i) c->sym_key[i] = -1;
    for (int i = 0; i < 16; ++i) c->smem_set[i] = 0;
    c->use_sym = 1;   // bie_set_symmetric
    c->small_gmres = 1; c->cluster_size = 0;   // bie_set_small_gmres; the cluster size is probed at the first small solve
    if (cudaMalloc((void**)&c->sync_buf, 256 * (BIE_SYNC_SLOTS + 1)) != cudaSuccess ||
        cudaMallocHost((void**)&c->pinned_i, 4 * sizeof(int32_t)) != cudaSuccess ||
        cudaMallocHost((void**)&c->pinned_d, 4 * sizeof(double)) != cudaSuccess) {
        cudaError_t le = cudaGetLastError();
        if (c->sync_buf) cudaFree(c->sync_buf);
        if (c->pinned_i) cudaFreeHost(c->pinned_i);
        delete c;
        return bie_cuda_err(le == cudaSuccess ? cudaErrorMemoryAllocation : le);
    }
    // the last 256-byte block holds a device scalar
    c->taubar = reinterpret_cast<double*>(reinterpret_cast<char*>(c->sync_buf) + 256 * BIE_SYNC_SLOTS);
    *out = c;
    return BIE_OK;
}

int bie_destroy(bie_ctx* c)
{
    if (!c) return BIE_ERR_NULL;
    cudaSetDevice(c->device);
    if (c->node_buf) cudaFree(c->node_buf);
    if (c->comp_buf) cudaFree(c->comp_buf);
    if (c->free_buf) cudaFree(c->free_buf);
    if (c->near_ptr) cudaFree(c->near_ptr);
    if (c->near_col) cudaFree(c->near_col);
    if (c->near_val) cudaFree(c->near_val);
    if (c->kappa) cudaFree(c->kappa);
    if (c->pc_buf) cudaFree(c->pc_buf);
    if (c->sym_tab) cudaFree(c->sym_tab);
    if (c->sync_buf) cudaFree(c->sync_buf);
    if (c->pinned_i) cudaFreeHost(c->pinned_i);
    if (c->pinned_d) cudaFreeHost(c->pinned_d);
    delete c;
    return BIE_OK;
}

const char* bie_strerror(int code)
{
    switch (code) {
        case BIE_OK: return "ok";
        case BIE_MAX_ITERS: return "max_iters reached before the residual test passed";
        case BIE_ERR_NULL: return "a required pointer is NULL";
        case BIE_ERR_GEOMETRY: return "bad geometry (ncomp/counts/kinds) or no geometry set";
        case BIE_ERR_LAYOUT: return "bad layout (lda < n, lda odd, or pointer not 16-byte aligned)";
        case BIE_ERR_WORKSPACE: return "workspace too small";
        case BIE_ERR_DEVICE: return "no usable compute-capability-10.x device";
        case BIE_ERR_ARG: return "bad argument";
        case BIE_ERR_NOALLOC_SIZE: return "bie_gmres_noalloc: (n, restart) needs more workspace than the static scratch (BIE_NOALLOC_SCRATCH_BYTES)";
        default: return code <= BIE_ERR_CUDA_BASE ? "CUDA runtime error (code = -100 - cudaError_t)" : "unknown code";
    }
}

int bie_device_info(bie_ctx* c, int* sm_count, int* fp64_fma_per_sm_clk, int* l2_bytes_mib)
{
    if (!c) return BIE_ERR_NULL;
    if (sm_count) *sm_count = c->sm_count;
    if (fp64_fma_per_sm_clk) *fp64_fma_per_sm_clk = 64;
    if (l2_bytes_mib) *l2_bytes_mib = c->l2_bytes >> 20;
    return BIE_OK;
}

int bie_set_geometry(bie_ctx* c, int ncomp, const int32_t* counts, const int32_t* kinds, const double* zeta,
                     const double* dzeta, const double* d2zeta, int variant, void* stream)
{
    if (!c) return BIE_ERR_NULL;
    if (variant < BIE_VARIANT_A || variant > BIE_VARIANT_VORTEX) return BIE_ERR_ARG;
    BIE_CUDA(cudaSetDevice(c->device));
    return bie_prepare_nodes(c, ncomp, counts, kinds, zeta, dzeta, d2zeta, variant, (cudaStream_t)stream);
}

int bie_build(bie_ctx* c, int ncomp, const int32_t* counts, const int32_t* kinds, const double* zeta,
              const double* dzeta, const double* d2zeta, int variant, double* A, int64_t lda, void* stream)
{
    if (variant < BIE_VARIANT_A || variant > BIE_VARIANT_VORTEX) return BIE_ERR_ARG;
    if (!c || !A) return BIE_ERR_NULL;
    BIE_CUDA(cudaSetDevice(c->device));
    int rc = bie_prepare_nodes(c, ncomp, counts, kinds, zeta, dzeta, d2zeta, variant, (cudaStream_t)stream);
    if (rc != BIE_OK) return rc;
    return bie_launch_build(c, A, lda, c->n, 0, 0, (cudaStream_t)stream);
}

int bie_build_update(bie_ctx* c, int ncomp, const int32_t* counts, const int32_t* kinds, const double* zeta,
                     const double* dzeta, const double* d2zeta, int variant, double* A, int64_t lda, void* stream)
{
    if (variant < BIE_VARIANT_A || variant > BIE_VARIANT_VORTEX) return BIE_ERR_ARG;
    if (!c || !A) return BIE_ERR_NULL;
    BIE_CUDA(cudaSetDevice(c->device));
    int rc = bie_prepare_nodes(c, ncomp, counts, kinds, zeta, dzeta, d2zeta, variant, (cudaStream_t)stream);
    if (rc != BIE_OK) return rc;
    return bie_launch_build(c, A, lda, c->n, 0, 1, (cudaStream_t)stream);
}

int bie_build_cols(bie_ctx* c, int ncomp, const int32_t* counts, const int32_t* kinds, const double* zeta,
                   const double* dzeta, const double* d2zeta, int variant, int ncols, double* A, int64_t lda, void* stream)
{
    if (variant < BIE_VARIANT_A || variant > BIE_VARIANT_VORTEX) return BIE_ERR_ARG;
    if (!c || !A) return BIE_ERR_NULL;
    BIE_CUDA(cudaSetDevice(c->device));
    int rc = bie_prepare_nodes(c, ncomp, counts, kinds, zeta, dzeta, d2zeta, variant, (cudaStream_t)stream);
    if (rc != BIE_OK) return rc;
    return bie_launch_build(c, A, lda, ncols, 0, 0, (cudaStream_t)stream);
}

// edge of the stored leading block of the hybrid operator: the share of n that makes the block stream and the pair loops
// finish together on a B200 (measured), rounded down to a row-block boundary of the pair
// loops: a multiple of 128 up to M_0, or M_0 plus a multiple of 128; even; 0 = too small to be worth it
static int hybrid_cols(int n, int M0)
{
    if (n < 4) return 0;
    if (M0 < 1 || M0 > n) M0 = n;
    const int target = (int)((double)n * BIE_HYBRID_DENSE_FRACTION);
    int nd = target <= M0 ? (target & ~127) : M0 + ((target - M0) & ~127);
    if (nd & 1) nd = M0 & ~127;      // M_0 odd: stay on Gamma_0
    if (nd < 128) nd = 0;
    if (nd > n - 2) nd = 0;
    return nd;
}

int bie_hybrid_cols(bie_ctx* c, int n)
{
    if (!c) return 0;
    return hybrid_cols(n, (c->have_geom && c->n == n) ? c->counts[0] : n);
}

size_t bie_hybrid_block_bytes(int nblock) { return nblock < 1 ? 0 : sizeof(double) * bie_block_doubles(nblock); }

int bie_build_block(bie_ctx* c, int ncomp, const int32_t* counts, const int32_t* kinds, const double* zeta,
                    const double* dzeta, const double* d2zeta, int variant, int nblock, double* A, void* stream)
{
    if (variant < BIE_VARIANT_A || variant > BIE_VARIANT_VORTEX) return BIE_ERR_ARG;
    if (!c || !A) return BIE_ERR_NULL;
    if (nblock < 1) return BIE_ERR_ARG;
    BIE_CUDA(cudaSetDevice(c->device));
    int rc = bie_prepare_nodes(c, ncomp, counts, kinds, zeta, dzeta, d2zeta, variant, (cudaStream_t)stream);
    if (rc != BIE_OK) return rc;
    return bie_launch_build(c, A, 0 /* block format */, nblock, nblock, 0, (cudaStream_t)stream);
}

int bie_set_symmetric(bie_ctx* c, int on)
{
    if (!c) return BIE_ERR_NULL;
    if (on < 0 || on > 2) return BIE_ERR_ARG;
    if ((c->use_sym != 0) != (on != 0)) c->near_valid = 0;   // the near matrix stores corrections for one or the other
    c->use_sym = on;
    return BIE_OK;
}

int bie_set_small_gmres(bie_ctx* c, int on)
{
    if (!c) return BIE_ERR_NULL;
    if (on < 0 || on > 1) return BIE_ERR_ARG;
    c->small_gmres = on;
    return BIE_OK;
}

int bie_set_hybrid_free_warps(bie_ctx* c, int free_warps)
{
    if (!c) return BIE_ERR_NULL;
    if (free_warps < 1 || free_warps > 15) return BIE_ERR_ARG;
    c->hybrid_free_warps = free_warps;
    return BIE_OK;
}

int bie_set_hybrid_poll_tiles(bie_ctx* c, int tiles)
{
    if (!c) return BIE_ERR_NULL;
    if (tiles < 0 || tiles > 64) return BIE_ERR_ARG;
    c->hybrid_poll_tiles = tiles;
    return BIE_OK;
}

int bie_matvec(bie_ctx* c, int n, const double* A, int64_t lda, const double* x, double* y, void* stream)
{
    if (!c) return BIE_ERR_NULL;
    BIE_CUDA(cudaSetDevice(c->device));
    return bie_launch_matvec(c, n, n, A, lda, x, y, (cudaStream_t)stream);
}

int bie_add_cyl_columns(bie_ctx* c, int ncomp, const int32_t* counts, const int32_t* kinds, const double* zeta,
                        const double* centers, double* A, int64_t lda, void* stream)
{
    if (!c) return BIE_ERR_NULL;
    BIE_CUDA(cudaSetDevice(c->device));
    return bie_launch_add_cyl_columns(c, ncomp, counts, kinds, zeta, centers, A, lda, (cudaStream_t)stream);
}

size_t bie_cauchy_eval_workspace_bytes(bie_ctx* c, int nf, int npts)
{
    return c ? bie_cauchy_eval_ws_bytes(nf, npts, c->sm_count) : 0;
}

int bie_cauchy_eval(bie_ctx* c, int ncomp, const int32_t* counts, const int32_t* kinds, const double* zeta,
                    const double* dzeta, int nf, const double* fvals, int npts, const double* zpts, double* out,
                    void* workspace, size_t workspace_bytes, void* stream)
{
    if (!c) return BIE_ERR_NULL;
    BIE_CUDA(cudaSetDevice(c->device));
    return bie_launch_cauchy_eval(c, ncomp, counts, kinds, zeta, dzeta, nf, fvals, npts, zpts, out, workspace,
                                  workspace_bytes, (cudaStream_t)stream);
}

int bie_matvec_rect(bie_ctx* c, int nrows, int ncols, const double* A, int64_t lda, const double* x, double* y,
                    void* stream)
{
    if (!c) return BIE_ERR_NULL;
    BIE_CUDA(cudaSetDevice(c->device));
    return bie_launch_matvec(c, nrows, ncols, A, lda, x, y, (cudaStream_t)stream);
}

int bie_build_normal_velocity(bie_ctx* c, int ncomp, const int32_t* counts, const int32_t* kinds, const double* zeta,
                              const double* dzeta, const double* d2zeta, double* Nmat, int64_t lda, void* stream)
{
    if (!c || !Nmat) return BIE_ERR_NULL;
    BIE_CUDA(cudaSetDevice(c->device));
    int rc = bie_prepare_nodes(c, ncomp, counts, kinds, zeta, dzeta, d2zeta, BIE_VARIANT_NORMAL_INTERNAL,
                               (cudaStream_t)stream);
    if (rc != BIE_OK) return rc;
    return bie_launch_build(c, Nmat, lda, c->n, 0, 0, (cudaStream_t)stream);
}

int bie_matvec_free(bie_ctx* c, int n, const double* x, double* y, void* stream)
{
    if (!c) return BIE_ERR_NULL;
    if (!c->have_geom || n != c->n) return BIE_ERR_GEOMETRY;
    BIE_CUDA(cudaSetDevice(c->device));
    return bie_launch_matvec_free(c, x, y, (cudaStream_t)stream);
}

size_t bie_gmres_workspace_bytes(int n, int restart) { return bie_gmres_ws_bytes(n, restart); }

int bie_gmres(bie_ctx* c, int n, const double* A, int64_t lda, const double* rhs, double tol, int restart,
              int max_iters, double* x, int32_t* iters_out, double* relres_out, int32_t* status_out,
              double* res_hist, void* workspace, size_t workspace_bytes, void* stream)
{
    if (!c) return BIE_ERR_NULL;
    BIE_CUDA(cudaSetDevice(c->device));
    return bie_launch_gmres(c, n, A, lda, 0, rhs, tol, restart, max_iters, x, iters_out, relres_out, status_out,
                            res_hist, workspace, workspace_bytes, (cudaStream_t)stream);
}

int bie_gmres_hybrid(bie_ctx* c, int n, const double* A, int ncols_dense, const double* rhs, double tol,
                     int restart, int max_iters, double* x, int32_t* iters_out, double* relres_out,
                     int32_t* status_out, double* res_hist, void* workspace, size_t workspace_bytes, void* stream)
{
    if (!c) return BIE_ERR_NULL;
    if (!A) return BIE_ERR_NULL;
    if (ncols_dense < 2) return BIE_ERR_ARG;
    BIE_CUDA(cudaSetDevice(c->device));
    return bie_launch_gmres(c, n, A, 0, ncols_dense, rhs, tol, restart, max_iters, x, iters_out, relres_out,
                            status_out, res_hist, workspace, workspace_bytes, (cudaStream_t)stream);
}

// ---- end-to-end with host buffers --------------------------------------------------------------------
static inline size_t up256(size_t b) { return (b + 255) & ~(size_t)255; }

// edge of bie_solve_host's stored part for an operator mode (dense: n, matrix-free: 0, hybrid: the leading block).
// Without the geometry (workspace query) the hybrid block is bounded by what any M_0 can give.
static int solve_cols(int n, int M0, int op)
{
    if (op == BIE_OP_FREE) return 0;
    if (op == BIE_OP_HYBRID) return hybrid_cols(n, M0);
    return n;
}

size_t bie_solve_workspace_bytes(int n, int restart, int matrix_free)
{
    if (n < 1 || restart < 1) return 0;
    // hybrid: the block edge depends on M_0; (frac n + 128)^2 bounds every case
    const size_t nblk = matrix_free == BIE_OP_HYBRID ? (size_t)((double)n * BIE_HYBRID_DENSE_FRACTION) + 130 : (size_t)solve_cols(n, n, matrix_free);
    const size_t nld = (nblk + 1) & ~(size_t)1;
    const size_t nvec = ((size_t)n + 1) & ~(size_t)1;
    size_t o = 256;
    o += 3 * up256(16 * (size_t)n);          // zeta, dzeta, d2zeta
    o += 2 * up256(8 * nvec);                // rhs, x
    o += up256(64);                          // iters, status, relres
    if (nld) o += up256(matrix_free == BIE_OP_HYBRID ? sizeof(double) * bie_block_doubles((int)nld) : 8 * nld * (size_t)n);
    o += bie_gmres_ws_bytes(n, restart);
    return o;
}

int bie_solve_host(bie_ctx* c, int ncomp, const int32_t* counts, const int32_t* kinds, const double* zeta,
                   const double* dzeta, const double* d2zeta, const double* rhs, double tol, int restart,
                   int max_iters, int matrix_free, double* x, int32_t* iters_out, double* relres_out,
                   void* dev_workspace, size_t dev_workspace_bytes, void* stream)
{
    if (!c || !counts || !kinds || !zeta || !dzeta || !d2zeta || !rhs || !x || !dev_workspace) return BIE_ERR_NULL;
    if (ncomp < 1 || ncomp > BIE_MAX_COMP) return BIE_ERR_GEOMETRY;
    long long nn = 0;
    for (int k = 0; k < ncomp; ++k) { if (counts[k] < 1) return BIE_ERR_GEOMETRY; nn += counts[k]; }
    if (nn > (1 << 30)) return BIE_ERR_GEOMETRY;
    if (restart < 1 || matrix_free < 0 || matrix_free > 2) return BIE_ERR_ARG;
    const int n = (int)nn;
    if (bie_solve_workspace_bytes(n, restart, matrix_free) > dev_workspace_bytes) return BIE_ERR_WORKSPACE;
    int ncols = solve_cols(n, counts[0], matrix_free);   // stored columns: n (dense), 0 (matrix-free), block edge (hybrid)
    if (matrix_free == BIE_OP_HYBRID && ncols == 0) { matrix_free = BIE_OP_FREE; }   // too small for a block: matrix-free
    const int nrows_st = matrix_free == BIE_OP_HYBRID ? ncols : n;                      // stored rows
    BIE_CUDA(cudaSetDevice(c->device));
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nld = ((size_t)ncols + 1) & ~(size_t)1;
    const size_t nvec = ((size_t)n + 1) & ~(size_t)1;
    char* p = (char*)(((uintptr_t)dev_workspace + 255) & ~(uintptr_t)255);
    double* dz0 = (double*)p; p += up256(16 * (size_t)n);
    double* dz1 = (double*)p; p += up256(16 * (size_t)n);
    double* dz2 = (double*)p; p += up256(16 * (size_t)n);
    double* drhs = (double*)p; p += up256(8 * nvec);
    double* dx = (double*)p; p += up256(8 * nvec);
    int32_t* dint = (int32_t*)p; double* drel = (double*)(p + 16); p += up256(64);
    double* dA = nullptr;
    const bool blockfmt = (matrix_free == BIE_OP_HYBRID);
    if (ncols) { dA = (double*)p; p += up256(blockfmt ? sizeof(double) * bie_block_doubles(ncols) : 8 * nld * (size_t)nrows_st); }
    void* gws = p;
    const size_t gws_bytes = bie_gmres_ws_bytes(n, restart);
    BIE_CUDA(cudaMemcpyAsync(dz0, zeta, 16 * (size_t)n, cudaMemcpyHostToDevice, st));
    BIE_CUDA(cudaMemcpyAsync(dz1, dzeta, 16 * (size_t)n, cudaMemcpyHostToDevice, st));
    BIE_CUDA(cudaMemcpyAsync(dz2, d2zeta, 16 * (size_t)n, cudaMemcpyHostToDevice, st));
    BIE_CUDA(cudaMemcpyAsync(drhs, rhs, 8 * (size_t)n, cudaMemcpyHostToDevice, st));
    int rc = bie_prepare_nodes(c, ncomp, counts, kinds, dz0, dz1, dz2, BIE_VARIANT_A, st);
    if (rc != BIE_OK) return rc;
    if (ncols) {
        rc = bie_launch_build(c, dA, blockfmt ? 0 : (int64_t)nld, ncols, nrows_st, 0, st);
        if (rc != BIE_OK) return rc;
    }
    rc = bie_launch_gmres(c, n, dA, (int64_t)nld, ncols < n ? ncols : 0, drhs, tol, restart, max_iters, dx, dint, drel,
                          dint + 1, nullptr, gws, gws_bytes, st);
    if (rc != BIE_OK) return rc;
    BIE_CUDA(cudaMemcpyAsync(x, dx, 8 * (size_t)n, cudaMemcpyDeviceToHost, st));
    BIE_CUDA(cudaMemcpyAsync(c->pinned_i, dint, 2 * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    BIE_CUDA(cudaMemcpyAsync(c->pinned_d, drel, sizeof(double), cudaMemcpyDeviceToHost, st));
    BIE_CUDA(cudaStreamSynchronize(st));
    if (iters_out) *iters_out = c->pinned_i[0];
    if (relres_out) *relres_out = c->pinned_d[0];
    return c->pinned_i[1] == BIE_MAX_ITERS ? BIE_MAX_ITERS : BIE_OK;
}

// ---- DFMA probe ------------------------------------------------------------------------------------------
}  // extern "C"

__global__ void __launch_bounds__(256) bie_probe_dfma_kernel(long long iters, double* out)
{
    // 8 independent chains per thread: the FP64 pipe is never latency-bound at 8 warps per scheduler
    double a0 = 1.0 + threadIdx.x * 1e-9, a1 = a0 + 1e-3, a2 = a0 + 2e-3, a3 = a0 + 3e-3;
    double a4 = a0 + 4e-3, a5 = a0 + 5e-3, a6 = a0 + 6e-3, a7 = a0 + 7e-3;
    const double m = 0.999999, c = 1e-7;
    for (long long i = 0; i < iters; ++i) {
        a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
        a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
    const double s = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (s == 12345.678) out[0] = s;  // never true; keeps the chains alive
}

int bie_launch_probe_dfma(bie_ctx* c, int64_t fma_per_thread, double* out, int64_t* total_fma, cudaStream_t st)
{
    if (!c || !out) return BIE_ERR_NULL;
    if (fma_per_thread < 8) return BIE_ERR_ARG;
    const long long iters = fma_per_thread / 8;
    const int blocks = c->sm_count * 8;  // 8 CTAs x 256 threads = 2048 threads per SM
    bie_probe_dfma_kernel<<<blocks, 256, 0, st>>>(iters, out);
    BIE_CUDA(cudaGetLastError());
    if (total_fma) *total_fma = (int64_t)iters * 8 * 256 * blocks;
    return BIE_OK;
}

// read-only streaming probe: every thread sums 128-bit evict-first loads of a buffer (what a GEMV does to its matrix)
__global__ void __launch_bounds__(512) bie_probe_read_kernel(const double2* __restrict__ p, long long n2, double* out)
{
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + 3 * stride < n2; i += 4 * stride) {
        const double2 v0 = __ldcs(p + i), v1 = __ldcs(p + i + stride), v2 = __ldcs(p + i + 2 * stride), v3 = __ldcs(p + i + 3 * stride);
        a0 += v0.x + v0.y; a1 += v1.x + v1.y; a2 += v2.x + v2.y; a3 += v3.x + v3.y;
    }
    for (; i < n2; i += stride) { const double2 v = __ldcs(p + i); a0 += v.x + v.y; }
    const double s = (a0 + a1) + (a2 + a3);
    if (s == 12345.678) out[0] = s;   // never true for the buffers bench.py passes; keeps the loads alive
}

extern "C" int bie_probe_read(bie_ctx* c, const double* buf, int64_t nbytes, double* out, void* stream)
{
    if (!c || !buf || !out) return BIE_ERR_NULL;
    if (nbytes < 16 || (((uintptr_t)buf) & 15u)) return BIE_ERR_LAYOUT;
    BIE_CUDA(cudaSetDevice(c->device));
    bie_probe_read_kernel<<<c->sm_count * 4, 512, 0, (cudaStream_t)stream>>>((const double2*)buf, (long long)(nbytes / 16), out);
    BIE_CUDA(cudaGetLastError());
    return BIE_OK;
}

extern "C" int bie_probe_dfma(bie_ctx* c, int64_t fma_per_thread, double* out, int64_t* total_fma, void* stream)
{
    if (!c) return BIE_ERR_NULL;
    BIE_CUDA(cudaSetDevice(c->device));
    return bie_launch_probe_dfma(c, fma_per_thread, out, total_fma, (cudaStream_t)stream);
}
