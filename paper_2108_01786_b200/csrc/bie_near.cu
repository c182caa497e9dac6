// bie_near.cu -- near-pair correction of the matrix-free operator (bie_free.cuh), built once per geometry.
//
// The fast pair arithmetic (one exponential per node, bie_common.cuh) cancels for |w| = |zeta_s - zeta_t| -> 0.
// A pair is NEAR when den = |E_s - E_t|^2 < taubar M_t, i.e. |e^{iw} - 1|^2 < taubar ~ |w|^2, with
// taubar = max_s clamp(BIE_NEAR_C |q_s|) one number per geometry (<= 1e-2, so that |w| < 0.11 and the Laurent
// series of bie_cot_half_near is exact to rounding).  The pair loop of the operator leaves near pairs out by
// predication; their exact matrix entries -- Laurent series of cot for s != t, the analytic diagonal limit
// K_jj(a,a) = Im{zeta''/(2 zeta')} with the -+1/2 of Eq. (3.10) for s == t, both WITHOUT the
// rank-one -E_k of PAPER.md:L324, which the operator applies through component sums, and (Eq. (3.16) variants) PLUS the
// constant beta_s of the difference form, which the operator subtracts for ALL sources at once (bie_free.cuh) -- are
// stored here as a sparse matrix in CSR form (a handful of entries per row: the neighbours on the same curve and whatever
// other curve comes closer than sqrt(taubar)), and added as  y_t += sum_k val[k] x[col[k]]  when the operator
// gathers its partial sums.  Classification uses exactly the expression of the pair loop, so both agree bit
// for bit.  Three launches per geometry: count, exclusive scan, fill (the first and last scan all n^2 pairs
// with 4 FP64 instructions each).  The arrays are sized from the scanned total (the host reads it back once per
// geometry and grows them on demand), so there is no capacity limit.
#include "bie_common.cuh"

#define NEAR_THREADS 128
#define NEAR_SEG 8          // source segments per target row: (row, segment) lists are contiguous in CSR order
#define NEAR_TILE 512

template <bool FILL>
__global__ void __launch_bounds__(NEAR_THREADS)
bie_near_kernel(NodeTable nt, CompTable ct, int vortex, int sym /* 1: pairs of different row blocks store exact - fast */,
                const double* __restrict__ taubar, int* __restrict__ cnt /* [n][NEAR_SEG] counts or offsets */,
                int* __restrict__ col, double* __restrict__ val, int cap)
{
    __shared__ double2 sE[NEAR_TILE];
    const int n = nt.n;
    const int t = blockIdx.x * NEAR_THREADS + threadIdx.x;
    const int seg = blockIdx.y;
    const int per = (nt.npad / NEAR_SEG + 1) & ~1;
    const int s_lo = seg * per, s_hi = min(s_lo + per, n);
    const int tt = min(t, n - 1);
    const double2 te = nt.E[tt];
    const int thi = __double2hiint(taubar[0] * nt.MT[tt].x);
    const bool tgt0 = (nt.COMP[tt] == 0);
    int k = 0, base = 0;
    if (FILL && t < n) base = cnt[(size_t)t * NEAR_SEG + seg];
    for (int s0 = s_lo; s0 < s_hi; s0 += NEAR_TILE) {
        __syncthreads();
        for (int i = threadIdx.x; i < NEAR_TILE; i += NEAR_THREADS)
            sE[i] = (s0 + i < s_hi) ? nt.E[s0 + i] : make_double2(0.0, 0.0);  // E = 0 is never near (den = M_t)
        __syncthreads();
        const int m = min(NEAR_TILE, s_hi - s0);
#pragma unroll 4
        for (int j = 0; j < m; ++j) {
            const double2 e = sE[j];
            const double dr = e.x - te.x, di = e.y - te.y;
            const double den = fma(dr, dr, di * di);
            if (__double2hiint(den) < thi) {
                if (FILL && t < n) {
                    const int s = s0 + j;
                    const int p = base + k;
                    if (p < cap) {   // always true: cap >= the scanned total
                        const double2 q = nt.Q[s];
                        const int jc = nt.COMP[s];
                        const bool src0 = (jc == 0);
                        double al, be;
                        if (src0 == tgt0) { al = -2.0 * q.y; be = q.x; }        // Im c     block coefficients of Eq. (3.10)
                        else if (tgt0)    { al = -2.0 * q.x; be = -q.y; }       // Re c   (G_0j)
                        else              { al = 2.0 * q.x;  be = q.y; }        // -Re c  (-G_k0)
                        double v;
                        if (s == t) {
                            const double2 dg = nt.DG[t];
                            v = dg.x + dg.y;   // complete diagonal entry without its -E_k part
                        } else {
                            const double2 zs = nt.XY[s], zt = nt.XY[t];
                            double cr, ci;
                            bie_cot_half_near(zs.x - zt.x, zs.y - zt.y, &cr, &ci);
                            if (vortex) {   // S of Eqs. (4.14) + (4.17): weight zeta'_t/2 of the ROW, 1/M_j of the column
                                const int kc = nt.COMP[t];
                                const double2 qt = nt.Q[t];
                                const double Mk = (double)(ct.off[kc + 1] - ct.off[kc]), ms = 1.0 / (double)(ct.off[jc + 1] - ct.off[jc]);
                                const double ur = qt.x * Mk * ms, ui = qt.y * Mk * ms;
                                if (src0 == tgt0) { al = 2.0 * ui;  be = -ur; }      // Im c+
                                else if (tgt0)    { al = -2.0 * ur; be = -ui; }      // -Re c+ (-G+_j0)
                                else              { al = 2.0 * ur;  be = ui; }       // Re c+  (G+_0k)
                            }
                            v = fma(be, ci, -0.5 * al * cr);   // cot = (-2X + iY)/den
                        }
                        if (!vortex) v += be;   // the operator subtracts sum_s beta_s x_s over ALL sources (difference form)
                        if (sym && s != t) {
                            // the symmetric pair loops (bie_free_sym.cuh) test nothing outside a row block's own rows: they add the
                            // FAST value of this pair, and this entry corrects it.  Row blocks: 128 rows, cut per class at M_0.
                            const int M0 = ct.off[1];
                            const int bt = t < M0 ? t / 128 : (M0 + 127) / 128 + (t - M0) / 128;
                            const int bs = s < M0 ? s / 128 : (M0 + 127) / 128 + (s - M0) / 128;
                            if (bt != bs) {
                                const double2 es = nt.E[s];
                                const double u = fma(al, es.y, 2.0 * be * es.x), w = fma(-al, es.x, 2.0 * be * es.y);
                                v -= fma(w, di, u * dr) * bie_rcp3(den);
                            }
                        }
                        col[p] = s;
                        val[p] = v;
                    }
                }
                ++k;
            }
        }
    }
    if (!FILL && t < n) cnt[(size_t)t * NEAR_SEG + seg] = k;
}

// exclusive prefix sum of N ints in place (N a multiple of 4, a 16-byte aligned), total to a[N]; one CTA.
// Thread i owns a contiguous run of int4; the loads of a run are independent and unrolled (the run is read twice,
// from L2).
__global__ void __launch_bounds__(1024) bie_near_scan_kernel(int* __restrict__ a, int N)
{
    __shared__ int sums[1024];
    int4* a4 = reinterpret_cast<int4*>(a);
    const int N4 = N >> 2;
    const int per = (N4 + 1023) / 1024;
    const int lo = min((int)threadIdx.x * per, N4), hi = min(lo + per, N4);
    int s = 0;
#pragma unroll 8
    for (int i = lo; i < hi; ++i) {
        const int4 v = __ldcg(a4 + i);
        s += (v.x + v.y) + (v.z + v.w);
    }
    sums[threadIdx.x] = s;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {   // Hillis-Steele inclusive scan
        const int v = (threadIdx.x >= o) ? sums[threadIdx.x - o] : 0;
        __syncthreads();
        sums[threadIdx.x] += v;
        __syncthreads();
    }
    int run = sums[threadIdx.x] - s;
#pragma unroll 8
    for (int i = lo; i < hi; ++i) {
        const int4 v = __ldcg(a4 + i);
        int4 o;
        o.x = run; o.y = o.x + v.x; o.z = o.y + v.y; o.w = o.z + v.z;
        run = o.w + v.w;
        a4[i] = o;
    }
    if (threadIdx.x == 1023) a[N] = sums[1023];
}

// builds the CSR near matrix of the ctx's current geometry if it is not there yet (lazy: the dense path never
// needs it).  SYNCHRONISES the stream once per geometry: the total number of near pairs comes back to the host and
// near_col / near_val grow to it when needed.
int bie_ensure_near(bie_ctx* ctx, cudaStream_t st)
{
    if (!ctx->have_geom) return BIE_ERR_GEOMETRY;
    if (ctx->near_valid) return BIE_OK;
    const NodeTable nt = bie_node_table(ctx);
    const int n = ctx->n;
    const int vx = (ctx->variant == BIE_VARIANT_VORTEX) ? 1 : 0;
    const int sym = bie_uses_sym(ctx) ? 1 : 0;
    dim3 grid((n + NEAR_THREADS - 1) / NEAR_THREADS, NEAR_SEG);
    bie_near_kernel<false><<<grid, NEAR_THREADS, 0, st>>>(nt, ctx->comps, vx, sym, ctx->taubar, ctx->near_ptr, nullptr, nullptr, 0);
    bie_near_scan_kernel<<<1, 1024, 0, st>>>(ctx->near_ptr, n * NEAR_SEG);
    BIE_CUDA(cudaGetLastError());
    BIE_CUDA(cudaMemcpyAsync(ctx->pinned_i + 2, ctx->near_ptr + (size_t)n * NEAR_SEG, sizeof(int), cudaMemcpyDeviceToHost, st));
    BIE_CUDA(cudaStreamSynchronize(st));
    const size_t total = (size_t)ctx->pinned_i[2];
    if (total > ctx->near_cap) {
        if (ctx->near_col) cudaFree(ctx->near_col);
        if (ctx->near_val) cudaFree(ctx->near_val);
        ctx->near_col = nullptr; ctx->near_val = nullptr; ctx->near_cap = 0;
        const size_t cap = total + total / 4 + 1024;
        if (cap > (size_t)0x7fffffff) return BIE_ERR_GEOMETRY;
        BIE_CUDA(cudaMalloc((void**)&ctx->near_col, sizeof(int) * cap));
        BIE_CUDA(cudaMalloc((void**)&ctx->near_val, sizeof(double) * cap));
        ctx->near_cap = cap;
    }
    bie_near_kernel<true><<<grid, NEAR_THREADS, 0, st>>>(nt, ctx->comps, vx, sym, ctx->taubar, ctx->near_ptr, ctx->near_col, ctx->near_val,
                                                        (int)ctx->near_cap);
    BIE_CUDA(cudaGetLastError());
    ctx->near_valid = 1;
    return BIE_OK;
}
