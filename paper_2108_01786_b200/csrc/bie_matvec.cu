// bie_matvec.cu -- SURVEY 8(a) row a6 as stand-alone calls: y = A x from the stored matrix (HBM-bound,
// bie_gemv.cuh) and the matrix-free operator that recomputes the entries of Eq. (3.16) on the fly
// (FP64-bound, bie_free.cuh).  One CTA per SM, each owning a contiguous block of rows.
#include "bie_common.cuh"
#include "bie_gemv.cuh"
#include "bie_free.cuh"

#define MV_THREADS 512

template <bool STREAM, bool XS>
__global__ void __launch_bounds__(MV_THREADS, 1)
bie_matvec_kernel(const double* __restrict__ A, long long lda, int nrows, int n, int rows_per_cta, int chunk, int res_pairs,
                  const double* __restrict__ x, double* __restrict__ y)
{
    extern __shared__ __align__(16) double smem[];
    const int r0 = blockIdx.x * rows_per_cta;
    const int r1 = min(r0 + rows_per_cta, nrows);
    if (r0 >= r1) return;
    double* y_local = smem;
    double* part = y_local + ((rows_per_cta + 1) & ~1);
    double* xs = part + gemv_part_doubles(rows_per_cta, n, chunk);
    if (XS) {
        const int n2 = n >> 1;
        for (int i = threadIdx.x; i < n2; i += blockDim.x)
            reinterpret_cast<double2*>(xs)[i] = __ldg(reinterpret_cast<const double2*>(x) + i);
        if ((n & 1) && threadIdx.x == 0) xs[n - 1] = x[n - 1];
        __syncthreads();
    }
    bie_cta_gemv<STREAM, XS>(A, lda, n, r0, r1, chunk, XS ? xs : x, part, y_local, cta_team(), res_pairs);
    for (int r = threadIdx.x; r < r1 - r0; r += blockDim.x) y[r0 + r] = y_local[r];
}

template <bool STREAM, bool XS>
static int launch_mv(bie_ctx* ctx, int nrows, int n, const double* A, int64_t lda, const double* x, double* y,
                     int rows_per_cta, int chunk, int res_pairs, size_t smem, cudaStream_t st)
{
    auto k = bie_matvec_kernel<STREAM, XS>;
    const int rc = bie_grant_smem(ctx, 8 + (STREAM ? 2 : 0) + (XS ? 1 : 0), k, smem);
    if (rc != BIE_OK) return rc;
    const int grid = (nrows + rows_per_cta - 1) / rows_per_cta;
    k<<<grid, MV_THREADS, smem, st>>>(A, (long long)lda, nrows, n, rows_per_cta, chunk, res_pairs, x, y);
    BIE_CUDA(cudaGetLastError());
    return BIE_OK;
}

// y (nrows) = A (nrows x n, row-major, lda) x (n)
int bie_launch_matvec(bie_ctx* ctx, int nrows, int n, const double* A, int64_t lda, const double* x, double* y,
                      cudaStream_t st)
{
    if (!ctx || !A || !x || !y) return BIE_ERR_NULL;
    if (n < 1 || nrows < 1) return BIE_ERR_ARG;
    if (lda < n || (lda & 1) || ((((uintptr_t)A) | ((uintptr_t)x) | ((uintptr_t)y)) & 15u)) return BIE_ERR_LAYOUT;
    const int G = ctx->sm_count;
    const int rows_per_cta = (nrows + G - 1) / G;
    const int chunk = gemv_chunk(rows_per_cta, n, MV_THREADS / 32);
    const size_t base = sizeof(double) * (((rows_per_cta + 1) & ~1) + gemv_part_doubles(rows_per_cta, n, chunk));
    const bool xs = base + sizeof(double) * ((size_t)n + 2) <= (size_t)ctx->max_smem_optin;
    const size_t smem = base + (xs ? sizeof(double) * ((size_t)n + 2) : 0);
    if (smem > (size_t)ctx->max_smem_optin) return BIE_ERR_ARG;
    // matrices that cannot stay in L2 are streamed (evict-first) so that they do not displace x, y and
    // the Krylov basis; smaller ones are read with the default policy and stay L2-resident between calls
    const bool stream = (double)nrows * (double)lda * 8.0 > 0.6 * (double)ctx->l2_bytes;
    const int res_pairs = stream ? bie_gemv_resident_pairs(ctx->l2_bytes, nrows, (long long)lda, rows_per_cta, 0) : 0;
    if (stream) return xs ? launch_mv<true, true>(ctx, nrows, n, A, lda, x, y, rows_per_cta, chunk, res_pairs, smem, st)
                          : launch_mv<true, false>(ctx, nrows, n, A, lda, x, y, rows_per_cta, chunk, res_pairs, smem, st);
    return xs ? launch_mv<false, true>(ctx, nrows, n, A, lda, x, y, rows_per_cta, chunk, res_pairs, smem, st)
              : launch_mv<false, false>(ctx, nrows, n, A, lda, x, y, rows_per_cta, chunk, res_pairs, smem, st);
}

// ---------------------------------------------------------------------------------------------------
// matrix-free: one cooperative launch, three phases separated by grid barriers (bie_free.cuh)
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(FREE_THREADS, 1)
bie_matvec_free_kernel(NodeTable nt, CompTable ct, FreePlan fp, int rows_per_cta, const double* __restrict__ x,
                       double* __restrict__ y, unsigned int* sync)
{
    extern __shared__ __align__(16) double smem[];
    const int n = nt.n;
    const int r0 = min(blockIdx.x * rows_per_cta, n);
    const int r1 = min(r0 + rows_per_cta, n);
    double* scratch = smem;
    double* y_local = scratch + free_scratch_doubles(fp.vortex != 0, fp.sym != 0);
    unsigned int target = 0;
    free_write_tables(nt, ct, fp, r0, r1, x + r0, scratch);
    grid_barrier(sync, target);
    free_parts(nt, ct, fp, scratch, cta_team(), NoPoll());
    grid_barrier(sync, target);
    free_gather(nt, ct, fp, r0, r1, x, 1.0, scratch, y_local);
    for (int r = threadIdx.x; r < r1 - r0; r += blockDim.x) y[r0 + r] = y_local[r];
}

int bie_launch_matvec_free(bie_ctx* ctx, const double* x, double* y, cudaStream_t st)
{
    if (!ctx || !x || !y) return BIE_ERR_NULL;
    if (!ctx->have_geom) return BIE_ERR_GEOMETRY;
    if ((((uintptr_t)x) | ((uintptr_t)y)) & 15u) return BIE_ERR_LAYOUT;
    if (!ctx->coop_ok || ctx->sm_count > 256) return BIE_ERR_DEVICE;
    const int n = ctx->n;
    const int G = ctx->sm_count;
    const int rows_per_cta = (n + G - 1) / G;
    FreePlan fp;
    int rc = bie_ensure_near(ctx, st);
    if (rc != BIE_OK) return rc;
    rc = bie_free_plan(ctx, G, 0, &fp, st);
    if (rc != BIE_OK) return rc;
    const size_t smem = sizeof(double) * (size_t)(free_scratch_doubles(fp.vortex != 0, fp.sym != 0) + ((rows_per_cta + 1) & ~1));
    if (smem > (size_t)ctx->max_smem_optin) return BIE_ERR_ARG;
    rc = bie_grant_smem(ctx, 12, bie_matvec_free_kernel, smem);
    if (rc != BIE_OK) return rc;
    // the grid-barrier counter of THIS launch: the ctx cycles through BIE_SYNC_SLOTS counters, so that a later launch
    // never resets a counter an earlier one may still be spinning on (a ctx serves one stream at a time, include/bie.h)
    unsigned int* sync = ctx->sync_buf + 64 * (ctx->sync_next++ % BIE_SYNC_SLOTS);
    BIE_CUDA(cudaMemsetAsync(sync, 0, sizeof(unsigned int), st));
    NodeTable nt = bie_node_table(ctx);
    CompTable ct = ctx->comps;
    int rpc = rows_per_cta;
    void* params[] = {(void*)&nt, (void*)&ct, (void*)&fp, (void*)&rpc, (void*)&x, (void*)&y, (void*)&sync};
    BIE_CUDA(cudaLaunchCooperativeKernel((const void*)bie_matvec_free_kernel, dim3(G), dim3(FREE_THREADS), params, smem, st));
    return BIE_OK;
}
