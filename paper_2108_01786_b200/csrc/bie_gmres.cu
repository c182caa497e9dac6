// bie_gmres.cu -- SURVEY 8(a) rows a5-a10: restarted GMRES(m) (Saad & Schultz, ref. [38] cited at
// PAPER.md:L855; stopping rule behind i_max) as ONE persistent cooperative kernel.
//
// The paper ran the GEMV on the GPU and shipped every Krylov vector over PCIe to orthogonalise on the CPU
// (PAPER.md:L857).  Here nothing leaves the device: one CTA per SM owns a contiguous block R of rows of A and,
// with it, the same rows of every Krylov vector.  Arnoldi step j, with TWO grid barriers (three for the matrix-free
// and hybrid operators, whose partial sums cross CTAs):
//     y[R]  = A[R,:] u / hn'                 u = the vector the previous step left in `wbuf` (see below), hn' its norm;
//                                            bie_cta_gemv (HBM-bound), or the pair loops of bie_free.cuh (FP64-bound,
//                                            + one grid barrier), or both at once (hybrid operator)
//     s     = V_j^T y                        local dots over R, GRID BARRIER 1, fixed-order sum
//     w1    = y - V_j s                      first classical Gram-Schmidt pass;  w1[R] -> wbuf
//     h2    = V_j^T w1,  nu = ||w1||^2       local dots over R, GRID BARRIER 2, fixed-order sum
//     v_{j+1} = (w1 - V_j h2) / hn,  hn^2 = nu - ||h2||^2      second pass (CGS2); h = s - c/hn' + h2
// Two things keep this at two barriers.  (i) The norm of the twice-orthogonalised vector comes from Pythagoras,
// ||w1 - V h2||^2 = ||w1||^2 - ||h2||^2, in the SAME reduction as h2; h2 is a rounding-level correction, so nothing
// cancels (guard: if ||h2||^2 > 0.01 nu the step falls back to an explicit norm with one more barrier).  (ii) The next
// operator application does not wait for v_{j+1} to be exchanged: it is applied to u = w1, whose rows went to `wbuf`
// BEFORE barrier 2, and A v_{j+1} = (A w1 - A V_j h2)/hn = (A w1 - V_{j+1} c)/hn with c = Hbar_j h2 by the Arnoldi
// relation A V_j = V_{j+1} Hbar_j.  The term V_{j+1} c lies in the span of the basis, so the Gram-Schmidt pass removes
// it from the vector exactly as it would have; only the coefficients see it:  h_{.,j+1} = (V^T y)/hn - c/hn + h2.
// c is a rounding-level quantity (h2 ~ eps ||w||) times Hbar, so a single-precision copy of Hbar (packed, in shared
// memory) is ample.  Every CTA reduces the per-CTA partials in the same fixed order, so all CTAs hold bit-identical
// h, Givens rotations and residuals and take the same branch without further communication.  The Givens /
// least-squares part (a8) is a few hundred flops done redundantly by thread 0 of every CTA; CTA 0 keeps R and does
// the back-substitution (a9) at the end of a cycle.  The grid-barrier counter lives in the caller's workspace.
#include <cstring>
#include "bie_common.cuh"
#include "bie_gemv.cuh"
#include "bie_free.cuh"

#ifndef GM_THREADS
#define GM_THREADS 512
#endif
#define GM_WARPS (GM_THREADS / 32)
#ifndef GM_WIDE_FROM
#define GM_WIDE_FROM 0      // rows of a reduction from which reduce_partials takes its seven-row form (developer knob)
#endif

struct GmresArgs {
    const double* A;
    long long lda;
    int n;
    const double* b;
    double tol;
    int m;
    int max_iters;
    double* x;
    int32_t* iters_out;
    double* relres_out;
    int32_t* status_out;
    double* res_hist;  // [max_iters+1] recurrence residual / ||b|| after each step, or NULL
    double* V;     // [(m+1)][nld]
    double* wbuf;  // [nld]
    double* part;  // [3][m+2][G]
    double* R;     // [m][m+1]  column j at R + j*(m+1)
    double* yv;    // [m]
    unsigned int* sync;
    int nld;
    int rows_per_cta;
    int chunk;
    int VS;        // Krylov vectors 0..VS-1 keep this CTA's rows in shared memory; the others in V (global, L2)
    int nd;        // hybrid operator: the leading nd x nd block comes from the stored block A, everything else is recomputed
    int nwf;       // hybrid operator: warps 0..nwf-1 run the pair loops (and take tiles of the stored block in between), warps
                   // nwf..14 only take tiles, warp 15 issues the bulk copies
    int poll_tiles; // hybrid operator: tiles a pair-loop warp may take between two source chunks
    int brows;     // hybrid operator: rows of the stored block each CTA streams (a multiple of RING_ROWS)
    double* yd;    // hybrid operator: [nld] product of the stored block with x[0, nd), written by the CTAs that streamed the rows
    int res_pairs; // streaming GEMV: leading row pairs of every CTA block kept L2-resident (bie_gemv.cuh)
    int scratch_doubles;  // matrix-free scratch in shared memory (full, or the smaller one of the one-directional loops)
    NodeTable nt;
    CompTable ct;
    FreePlan fp;
};

// sum over the CTA; result to all threads.  red: shared, >= 33 doubles
__device__ __forceinline__ double block_sum(double v, double* red)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    v = bie_warp_sum(v);
    __syncthreads();
    if (lane == 0) red[warp] = v;
    __syncthreads();
    if (warp == 0) {
        double s = (lane < (int)(blockDim.x >> 5)) ? red[lane] : 0.0;
        s = bie_warp_sum(s);
        if (lane == 0) red[32] = s;
    }
    __syncthreads();
    return red[32];
}

// sum of the G per-CTA partials p[0..G), same order in every CTA; all lanes of the calling warp get it
__device__ __forceinline__ double warp_sum_partials(const double* p, int G)
{
    double s = 0.0;
    for (int c = threadIdx.x & 31; c < G; c += 32) s += __ldcg(p + c);
    return bie_warp_sum(s);
}

#ifdef BIE_PHASE_TIMING   // developer build (BIE_NVCC_EXTRA=-DBIE_PHASE_TIMING): three CTAs print the mean time per Arnoldi step of each phase
#include <cstdio>
__device__ __forceinline__ unsigned long long gtime() { unsigned long long t; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t)); return t; }
#ifndef BIE_PT_PAIR_ONLY
#define BIE_PT_PAIR_ONLY 0
#endif
__device__ unsigned long long g_pt[3][16];
__device__ unsigned long long g_pt0[3];
__device__ unsigned long long g_pair[256], g_gath[256];   // per CTA: accumulated pair-loop / gather time of the current cycle
__device__ __forceinline__ int pt_slot() { return blockIdx.x == 0 ? 0 : (blockIdx.x == gridDim.x / 2 ? 1 : (blockIdx.x == gridDim.x - 1 ? 2 : -1)); }
#define PT_RESET { if (threadIdx.x == 0) { g_pair[blockIdx.x] = 0; g_gath[blockIdx.x] = 0; } const int s_ = pt_slot(); if (threadIdx.x == 0 && s_ >= 0) { for (int q_ = 0; q_ < 16; ++q_) g_pt[s_][q_] = 0; g_pt0[s_] = gtime(); } }
#define PT(i) { const int s_ = pt_slot(); if (threadIdx.x == 0 && s_ >= 0) { const unsigned long long t_ = gtime(); g_pt[s_][i] += t_ - g_pt0[s_]; g_pt0[s_] = t_; } }
#else
#define PT_RESET
#define PT(i)
#endif

// MODE: 0 = stored matrix (GEMV, HBM-bound), 1 = matrix-free (pair loops, FP64-bound), 2 = hybrid: the leading
// nd x nd block is stored and arrives through the block ring of bie_gemv.cuh WHILE the warps recompute every other
// entry -- the HBM pipe and the FP64 pipe of every SM work at the same time.
template <bool STREAM, bool XS, int MODE>
__device__ __forceinline__ void cta_apply(const GmresArgs& a, int r0, int r1, const double* xin, double scale,
                                          double* xs, double* gpart, BlockRing& ring, double* y_local,
                                          bool tables_ready, double* red, unsigned int& target, int& sb_sel)
{
    if (MODE != 0) {
        // xin is complete in global memory; its per-source tables either were written by the row owners before
        // the last grid barrier (tables_ready) or are written here
        if (!tables_ready) {
            sb_sel ^= 1;
            free_write_tables(a.nt, a.ct, a.fp, r0, r1, xin + r0, red, sb_sel);
            grid_barrier(a.sync, target);
        }
        PT(6)
        if (MODE == 1) {
#ifdef BIE_PHASE_TIMING
            const unsigned long long tp0 = gtime();
#endif
            free_parts(a.nt, a.ct, a.fp, gpart, cta_team(), NoPoll());
#ifdef BIE_PHASE_TIMING
            if (threadIdx.x == 0) g_pair[blockIdx.x] += gtime() - tp0;
#endif
            PT(7)
        } else {
            const int warp = threadIdx.x >> 5;
            if (threadIdx.x == 0) { ring.next[0] = 0; ring.next[1] = 0; }
            __syncthreads();
            // nwf >= 12: the service warps -- the producer (warp 15) and 15 - nwf consumer warps -- all sit on ONE of the SM's
            // four sub-partitions (warp & 3 == 3: warps 15, 11, 7, 3), so that they do not wait for issue slots behind the
            // pair-loop warps of the other three.  nwf = 12: the pair loops run on exactly three sub-partitions, four warps
            // each, as in the matrix-free kernel.  nwf < 12: warps nwf..14 consume, wherever they sit.
            const bool split = (a.nwf >= 12);
            const int first_service = 3 + 4 * (a.nwf - 12);                     // split: service warps are first_service, +4, ..., 15
            const bool service = split ? ((warp & 3) == 3 && warp >= first_service) : (warp >= a.nwf);
            if (warp == GM_WARPS - 1) {
                if ((threadIdx.x & 31) == 0) ring_produce<STREAM>(ring, xin);
                __syncwarp();
            } else {
                if (!service) {
                    Team tm = sub_team(0, a.nwf, 1);
                    if (split) {   // index among the pair-loop warps: the service warps below this one do not count
                        tm.warp = warp - (warp > first_service ? ((warp - first_service + 3) >> 2) : 0);
                        tm.tid = 32 * tm.warp + (threadIdx.x & 31);
                    }
                    free_parts(a.nt, a.ct, a.fp, gpart, tm, RingPoll{&ring, a.poll_tiles});
                }
                while (ring_consume(ring)) { }
            }
            __syncthreads();
            // the rows of the stored block this CTA streamed: chunk sums in fixed order -> yd (their owners read it after the barrier)
            for (int r = threadIdx.x; r < ring.r1 - ring.r0; r += blockDim.x) {
                double sum = 0.0;
                for (int ch = 0; ch < ring.nch; ++ch) sum += ring.part[ch * ring.rowsP + r];
                a.yd[ring.r0 + r] = sum;
            }
            ring.tile0 += (unsigned long long)ring.nunit;
        }
        grid_barrier(a.sync, target);
        PT(8)
#ifdef BIE_PHASE_TIMING
        const unsigned long long tg0 = gtime();
#endif
        free_gather(a.nt, a.ct, a.fp, r0, r1, xin, scale, gpart, y_local, sb_sel);
#ifdef BIE_PHASE_TIMING
        if (threadIdx.x == 0) g_gath[blockIdx.x] += gtime() - tg0;
#endif
        PT(9)
        if (MODE == 2) {
            for (int r = threadIdx.x; r < r1 - r0; r += blockDim.x)
                if (r0 + r < a.nd) y_local[r] = fma(scale, __ldcg(a.yd + r0 + r), y_local[r]);
            __syncthreads();
        }
    } else if (XS) {
        const int n2 = a.n >> 1;
        for (int i = threadIdx.x; i < n2; i += blockDim.x) {
            double2 v = __ldcg(reinterpret_cast<const double2*>(xin) + i);
            v.x *= scale; v.y *= scale;
            reinterpret_cast<double2*>(xs)[i] = v;
        }
        if ((a.n & 1) && threadIdx.x == 0) xs[a.n - 1] = __ldcg(xin + a.n - 1) * scale;
        __syncthreads();
        bie_cta_gemv<STREAM, true>(a.A, a.lda, a.n, r0, r1, a.chunk, xs, gpart, y_local, cta_team(), a.res_pairs);
    } else {
        bie_cta_gemv<STREAM, false>(a.A, a.lda, a.n, r0, r1, a.chunk, xin, gpart, y_local, cta_team(), a.res_pairs);
        if (scale != 1.0) {
            for (int r = threadIdx.x; r < r1 - r0; r += blockDim.x) y_local[r] *= scale;
            __syncthreads();
        }
    }
}

// This CTA's rows of Krylov vector i: in shared memory for i < VS, else in the global basis (L2-resident).
struct Basis {
    double* Vs;      // shared, [VS][rows2]
    double* Vg;      // global, a.V + r0, vector stride nld
    int VS, rows2;
    long long nld;
};

// t[r] = sum_{i < cnt} coef[i] * v_i[r] for this CTA's rows, using every thread: the threads form `groups`
// groups of rp threads; group g takes the vectors i = g, g + groups, ...; the group sums are added in fixed
// order.  red2: shared, >= blockDim.x + rows2 doubles.  Result in red2[0 .. rows) after the closing barrier.
__device__ __forceinline__ void basis_combine(const Basis& B, int rows, int cnt, const double* coef, double* red2)
{
    int rp = (rows + 31) & ~31;
    if (rp > (int)blockDim.x) rp = blockDim.x;
    const int groups = blockDim.x / rp;
    const int g = threadIdx.x / rp, lr = threadIdx.x - g * rp;
    const int cs_ = min(cnt, B.VS);
    if (g < groups) {
        for (int r = lr; r < rows; r += rp) {
            double s0 = 0.0, s1 = 0.0;
            int i = g;
            const double* vs = B.Vs + r;
            for (; i + groups < cs_; i += 2 * groups) {
                s0 = fma(coef[i], vs[(size_t)i * B.rows2], s0);
                s1 = fma(coef[i + groups], vs[(size_t)(i + groups) * B.rows2], s1);
            }
            for (; i < cs_; i += groups) s0 = fma(coef[i], vs[(size_t)i * B.rows2], s0);
            const double* vg = B.Vg + r;
#pragma unroll 4
            for (; i < cnt; i += groups) s1 = fma(coef[i], __ldcg(vg + (size_t)i * B.nld), s1);
            red2[g * rp + r] = s0 + s1;   // rows <= rp unless groups == 1
        }
    }
    __syncthreads();
    if (groups > 1) {
        double t = 0.0;
        const int r = threadIdx.x;
        if (r < rows)
            for (int q = 0; q < groups; ++q) t += red2[q * rp + r];
        __syncthreads();
        if (r < rows) red2[r] = t;
        __syncthreads();
    }
}

// part_slot[i][cta] = <v_i, w>_R for i < cnt (this CTA's rows R); with_norm: part_slot[cnt][cta] = ||w||_R^2
__device__ __forceinline__ void local_dots(const Basis& B, int rows, int cnt, const double* w_local, double* part_slot,
                                           bool with_norm)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    const int G = gridDim.x;
    const int tot = cnt + (with_norm ? 1 : 0);
    // a warp takes TWO vectors at a time (i and i + nwarp): their loads and their lane reductions overlap
    for (int i = warp; i < tot; i += 2 * nwarp) {
        const int i2 = i + nwarp;
        const bool two = (i2 < tot);
        double s = 0.0, s2 = 0.0;
        const double* va = (i == cnt) ? w_local : ((i < B.VS) ? B.Vs + (size_t)i * B.rows2 : B.Vg + (size_t)i * B.nld);
        const double* vb = !two ? w_local : ((i2 == cnt) ? w_local : ((i2 < B.VS) ? B.Vs + (size_t)i2 * B.rows2 : B.Vg + (size_t)i2 * B.nld));
        const bool ga = (i != cnt && i >= B.VS), gb = (two && i2 != cnt && i2 >= B.VS);      // in the global basis (L2)
        for (int r = lane; r < rows; r += 32) {
            const double wr = w_local[r];
            const double a = ga ? __ldcg(va + r) : va[r];
            const double b = gb ? __ldcg(vb + r) : vb[r];
            s = fma(a, wr, s);
            s2 = fma(b, wr, s2);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            s += __shfl_xor_sync(0xffffffffu, s, o);
            s2 += __shfl_xor_sync(0xffffffffu, s2, o);
        }
        if (lane == 0) {
            part_slot[(size_t)i * G + blockIdx.x] = s;
            if (two) part_slot[(size_t)i2 * G + blockIdx.x] = s2;
        }
    }
}

// out[i] = sum over the G per-CTA partials of row i < cnt, same order in every CTA.  G even and <= 192 (one CTA per SM on a
// B200: 148): a row is at most three 128-bit loads per lane and a warp keeps SEVEN rows in flight, so that the restart + 2 <= 112
// rows of a reduction are ONE round of L2 latency for the 16 warps (four rows of 64-bit loads need two rounds from j = 63 on).
// Same box, A/B/A/B: config 5 26.66 -> 26.35 ms per solve, config 3 33.8 -> 31.9 us per iteration, config 2 0.597 -> 0.592 ms; taking
// this form only beyond 64 rows gives half of the gain.  Ends with __syncthreads.
__device__ __forceinline__ void reduce_partials(const double* part_slot, int cnt, double* out)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    const int G = gridDim.x;
    if ((G & 1) == 0 && G <= 192 && cnt > GM_WIDE_FROM) {
        constexpr int RP = 7;
        const int g2 = G >> 1;
        for (int i0 = warp; i0 < cnt; i0 += RP * nwarp) {
            double2 v[RP][3];
#pragma unroll
            for (int q = 0; q < RP; ++q) {
                const int i = i0 + q * nwarp;
                const double2* row = reinterpret_cast<const double2*>(part_slot + (size_t)i * G);
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    const int c = lane + 32 * k;
                    v[q][k] = (i < cnt && c < g2) ? __ldcg(row + c) : make_double2(0.0, 0.0);
                }
            }
            // the lane reductions of the rows in two interleaved groups (four and three rows; the second only if it has a row)
            double h[RP];
#pragma unroll
            for (int q = 0; q < RP; ++q) h[q] = ((v[q][0].x + v[q][0].y) + (v[q][1].x + v[q][1].y)) + (v[q][2].x + v[q][2].y);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
                for (int q = 0; q < 4; ++q) h[q] += __shfl_xor_sync(0xffffffffu, h[q], o);
            }
            if (i0 + 4 * nwarp < cnt) {                    // warp-uniform
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
                    for (int q = 4; q < RP; ++q) h[q] += __shfl_xor_sync(0xffffffffu, h[q], o);
                }
            }
#pragma unroll
            for (int q = 0; q < RP; ++q) {
                const int i = i0 + q * nwarp;
                if (i < cnt && lane == 0) out[i] = h[q];
            }
        }
        __syncthreads();
        return;
    }
    for (int i0 = warp; i0 < cnt; i0 += 4 * nwarp) {
        double s[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int i = i0 + q * nwarp;
            s[q] = 0.0;
            if (i < cnt)
                for (int c = lane; c < G; c += 32) s[q] += __ldcg(part_slot + (size_t)i * G + c);
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int i = i0 + q * nwarp;
            const double h = bie_warp_sum(s[q]);
            if (i < cnt && lane == 0) out[i] = h;
        }
    }
    __syncthreads();
}

// offset of column i of the packed upper-Hessenberg matrix (column i holds rows 0 .. i+1)
__device__ __forceinline__ int hess_off(int i) { return (i * (i + 3)) >> 1; }

// doubles of shared memory before the operator's scratch: y, w [rows2 each], hcol, hloc, cvec [m + 2 each], cs, sn [m each],
// g [m + 1], red [130], the packed single-precision Hbar [m (m + 3) / 2 floats]; rounded to 16 bytes
// + (matrix-free and hybrid operators) the per-source constants of this CTA's rows, [3][rows2] double2
__host__ __device__ inline int gm_head_doubles(int m, int rows2, bool free_op)
{
    int o = 2 * rows2 + 3 * (m + 2) + 2 * m + (m + 1) + 130;
    o += (m * (m + 3) / 2 + 1) / 2;
    o = (o + 1) & ~1;
    return o + (free_op ? 6 * rows2 : 0);
}

template <bool STREAM, bool XS, int MODE>
__global__ void __launch_bounds__(GM_THREADS, 1) bie_gmres_kernel(const GmresArgs a)
{
    constexpr bool FREE = (MODE != 0);
    extern __shared__ __align__(16) double smem[];
    const int G = gridDim.x;
    const int n = a.n, m = a.m;
    const int r0 = blockIdx.x * a.rows_per_cta;
    const int r1 = min(r0 + a.rows_per_cta, n);
    const int rows = r1 - r0;  // >= 1 by construction of the grid
    const int rows2 = (a.rows_per_cta + 1) & ~1;
    // shared layout
    double* y_local = smem;               // [rows2]   result of the operator
    double* w_local = y_local + rows2;    // [rows2]   the vector being orthogonalised
    double* hcol = w_local + rows2;       // [m+2]     column j of H
    double* hloc = hcol + (m + 2);        // [m+2]     coefficients of the current pass
    double* cvec = hloc + (m + 2);        // [m+2]     c = Hbar h2 of the previous step (see the header)
    double* cs = cvec + (m + 2);          // [m]
    double* sn = cs + m;                  // [m]
    double* g = sn + m;                   // [m+1]
    double* red = g + (m + 1);            // [130]
    float* Hf = reinterpret_cast<float*>(red + 130);                 // packed Hbar in single precision, m (m + 3) / 2 floats
    double* gpart = smem + gm_head_doubles(m, rows2, FREE);          // GEMV partials or matrix-free scratch (16-byte aligned)
    double2* Kc = reinterpret_cast<double2*>(gpart) - 3 * rows2;     // FREE: per-source constants of this CTA's rows
    // dense: GEMV partials, then x; matrix-free: the operator's scratch; hybrid: scratch, row sums of the ring's tiles, the ring
    double* ring_part = gpart + (FREE ? a.scratch_doubles : 0);
    double* ring_mem = ring_part + ((MODE == 2) ? ring_part_doubles(a.brows, a.nd, a.chunk) : 0);
    double* xs = gpart + ((MODE == 0) ? ((gemv_part_doubles(a.rows_per_cta, n, a.chunk) + 1) & ~1) : 0);
    double* red2 = (MODE == 2) ? ring_mem + ring_doubles(a.chunk)
                               : ((MODE == 1) ? ring_part : xs + (XS ? ((n + 2) & ~1) : 0));   // [blockDim + rows2]
    BlockRing ring;
    if (MODE == 2) {
        ring.A = a.A; ring.nd = a.nd; ring.chunk = a.chunk;
        ring.r0 = min(blockIdx.x * a.brows, a.nd); ring.r1 = min(ring.r0 + a.brows, a.nd);
        ring.nch = (a.nd + a.chunk - 1) / a.chunk;
        ring.nunit = ((ring.r1 - ring.r0 + RING_ROWS - 1) / RING_ROWS) * ring.nch;
        ring.stage = ring_mem;
        ring.full0 = smem_u32(ring_mem + RING_STAGES * (RING_ROWS + 1) * a.chunk);
        ring.empty0 = ring.full0 + 8 * RING_STAGES;
        ring.next = reinterpret_cast<int*>(ring_mem + RING_STAGES * (RING_ROWS + 1) * a.chunk + 2 * RING_STAGES);
        ring.part = ring_part;
        ring.rowsP = ((a.brows + RING_ROWS - 1) / RING_ROWS) * RING_ROWS;
        ring.tile0 = 0;
        ring_init(ring_mem, a.chunk);
    }
    Basis B;
    B.Vs = red2 + GM_THREADS + rows2;                          // [VS][rows2]
    B.Vg = a.V + r0; B.VS = a.VS; B.rows2 = rows2; B.nld = a.nld;
    if (FREE) free_init_row_consts(a.nt, a.ct, a.fp, r0, r1, Kc, rows2);
    double* part1 = a.part;
    double* part2 = a.part + (size_t)(m + 2) * G;
    double* part3 = a.part + 2 * (size_t)(m + 2) * G;
    unsigned int target = 0;

    // ---- a5: ||b||, x = 0 -------------------------------------------------------------------------
    double p = 0.0;
    for (int r = threadIdx.x; r < rows; r += blockDim.x) {
        const double v = a.b[r0 + r];
        p = fma(v, v, p);
        a.x[r0 + r] = 0.0;
    }
    p = block_sum(p, red);
    if (threadIdx.x == 0) part3[blockIdx.x] = p;
    grid_barrier(a.sync, target);
    const double bn = sqrt(warp_sum_partials(part3, G));
    const double thresh = a.tol * bn;

    int iters = 0, status = 0;
    bool done = (bn == 0.0);
    if (a.res_hist && blockIdx.x == 0 && threadIdx.x == 0) a.res_hist[0] = 1.0;
    bool first = true;
    // which copy of the constants' partials (FreePlan::SB) the last table write filled.  The copies alternate because the
    // table write at a cycle's start follows the gather of the residual's operator application WITHOUT a grid barrier in
    // between: a CTA that is done may write while others still read the previous copy.
    int sb_sel = 0;
    while (!done) {
        // ---- cycle start: r = b - A x ------------------------------------------------------------
        if (first) {
            for (int r = threadIdx.x; r < rows; r += blockDim.x) w_local[r] = a.b[r0 + r];
            first = false;
        } else {
            cta_apply<STREAM, XS, MODE>(a, r0, r1, a.x, 1.0, xs, gpart, ring, y_local, false, red, target, sb_sel);
            for (int r = threadIdx.x; r < rows; r += blockDim.x) w_local[r] = a.b[r0 + r] - y_local[r];
        }
        __syncthreads();
        p = 0.0;
        for (int r = threadIdx.x; r < rows; r += blockDim.x) {
            const double v = w_local[r];
            p = fma(v, v, p);
            a.wbuf[r0 + r] = v;
        }
        if (FREE) { sb_sel ^= 1; free_write_tables_cached(a.fp, a.nt.npad, r0, r1, w_local, Kc, rows2, red, sb_sel); }
        p = block_sum(p, red);
        if (threadIdx.x == 0) part3[blockIdx.x] = p;
        grid_barrier(a.sync, target);
        const double beta = sqrt(warp_sum_partials(part3, G));
        if (beta <= thresh) break;                         // converged (status 0)
        if (iters >= a.max_iters) { status = BIE_MAX_ITERS; break; }
        double inv = 1.0 / beta;                           // 1 / norm of the vector in wbuf
        {
            double* v0 = (0 < B.VS) ? B.Vs : B.Vg;
            for (int r = threadIdx.x; r < rows; r += blockDim.x) v0[r] = w_local[r] * inv;
        }
        for (int i = threadIdx.x; i < m + 2; i += blockDim.x) cvec[i] = 0.0;   // wbuf holds beta v_0 itself: no correction
        if (threadIdx.x == 0) g[0] = beta;
        __syncthreads();

        // ---- Arnoldi steps ------------------------------------------------------------------------
        int k = 0;
        bool conv = false;
        PT_RESET
        for (int j = 0; j < m; ++j) {
            PT(5)
            // a6: y = A (wbuf * inv) = A v_j + V_j c * inv  (c = 0 in the first step of a cycle)
            cta_apply<STREAM, XS, MODE>(a, r0, r1, a.wbuf, inv, xs, gpart, ring, y_local, true, red, target, sb_sel);
            PT(0)
            // a7, first pass: s = V_j^T y (grid barrier 1), w1 = y - V_j s, h1 = s - c * inv
            local_dots(B, rows, j + 1, y_local, part1, false);
            grid_barrier(a.sync, target);
            PT(1)
            reduce_partials(part1, j + 1, hloc);
            for (int i = threadIdx.x; i <= j; i += blockDim.x) hcol[i] = fma(-cvec[i], inv, hloc[i]);
            basis_combine(B, rows, j + 1, hloc, red2);
            for (int r = threadIdx.x; r < rows; r += blockDim.x) {
                const double v = y_local[r] - red2[r];
                w_local[r] = v;
                a.wbuf[r0 + r] = v;                       // the next operator application reads w1 (see the header)
            }
            __syncthreads();
            if (FREE) { sb_sel ^= 1; free_write_tables_cached(a.fp, a.nt.npad, r0, r1, w_local, Kc, rows2, red, sb_sel); }
            // second pass: h2 = V_j^T w1 and ||w1||^2 in ONE reduction (grid barrier 2)
            local_dots(B, rows, j + 1, w_local, part2, true);
            PT(2)
            grid_barrier(a.sync, target);
            PT(3)
            reduce_partials(part2, j + 2, hloc);          // hloc[0..j] = h2, hloc[j+1] = ||w1||^2
            if (threadIdx.x < 32) {                        // ||h2||^2, fixed order
                double ss = 0.0;
                for (int i = threadIdx.x; i <= j; i += 32) ss = fma(hloc[i], hloc[i], ss);
                ss = bie_warp_sum(ss);
                if (threadIdx.x == 0) red[128] = ss;
            }
            __syncthreads();
            PT(10)
            const double nu = hloc[j + 1], ss = red[128];
            double hn;
            const bool pyth = (ss <= 0.01 * nu);           // identical in every CTA (same bits)
            basis_combine(B, rows, j + 1, hloc, red2);     // V_j h2 on this CTA's rows
            if (pyth) {
                hn = sqrt(nu - ss);                        // ||w1 - V h2||^2 = ||w1||^2 - ||h2||^2, no cancellation: ss << nu
            } else {
                // w1 is NOT nearly orthogonal to the basis (breakdown region): explicit norm of w2 = w1 - V h2, and the
                // next operator application reads w2 (one more grid barrier; c = 0)
                p = 0.0;
                for (int r = threadIdx.x; r < rows; r += blockDim.x) {
                    const double v = w_local[r] - red2[r];
                    w_local[r] = v; red2[r] = 0.0;
                    p = fma(v, v, p);
                    a.wbuf[r0 + r] = v;
                }
                __syncthreads();
                if (FREE) { sb_sel ^= 1; free_write_tables_cached(a.fp, a.nt.npad, r0, r1, w_local, Kc, rows2, red, sb_sel); }
                p = block_sum(p, red);
                if (threadIdx.x == 0) part3[blockIdx.x] = p;
                grid_barrier(a.sync, target);
                hn = sqrt(warp_sum_partials(part3, G));
            }
            PT(11)
            inv = (hn != 0.0) ? 1.0 / hn : 0.0;
            {
                double* vn = (j + 1 < B.VS) ? B.Vs + (size_t)(j + 1) * rows2 : B.Vg + (size_t)(j + 1) * a.nld;
                for (int r = threadIdx.x; r < rows; r += blockDim.x) vn[r] = (w_local[r] - red2[r]) * inv;
            }
            for (int i = threadIdx.x; i <= j; i += blockDim.x) hcol[i] += hloc[i];
            __syncthreads();
            PT(12)
            // column j of Hbar (single precision copy), then c = Hbar_j h2 for the next step
            for (int i = threadIdx.x; i <= j + 1; i += blockDim.x) Hf[hess_off(j) + i] = (float)(i <= j ? hcol[i] : hn);
            __syncthreads();
            for (int t0 = 0; t0 < 4 * (j + 2); t0 += blockDim.x) {   // four threads per entry of c; whole warps take part
                const int t = t0 + threadIdx.x;
                if ((t & ~31) >= 4 * (j + 2)) continue;              // warp-uniform
                const int kk = t >> 2, q = t & 3;
                double c = 0.0;
                if (pyth && kk <= j + 1)
                    for (int i = max(kk - 1, 0) + q; i <= j; i += 4) c = fma((double)Hf[hess_off(i) + kk], hloc[i], c);
                c += __shfl_xor_sync(0xffffffffu, c, 1);
                c += __shfl_xor_sync(0xffffffffu, c, 2);
                if (q == 0 && kk <= j + 1) cvec[kk] = c;
            }
            PT(13)
            // a8: Givens rotations on column j, new rotation, recurrence residual
            if (threadIdx.x == GM_THREADS - 1) {
                hcol[j + 1] = hn;
                // rotation i maps (a, h_{i+1}) to (c a + s h_{i+1}, -s a + c h_{i+1}) and hands the second value on as the next a:
                // the products with the FRESH entry h_{i+1} are off the chain, which is one FMA per rotation
                // (blocks of four with all loads first: a store to hcol[i] would otherwise hold back the loads of the next rotation)
                double carry = hcol[0];
                int i = 0;
                for (; i + 4 <= j; i += 4) {
                    double c4[4], s4[4], h4[4], o4[4];
#pragma unroll
                    for (int q = 0; q < 4; ++q) { c4[q] = cs[i + q]; s4[q] = sn[i + q]; h4[q] = hcol[i + q + 1]; }
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        o4[q] = fma(c4[q], carry, s4[q] * h4[q]);
                        carry = fma(-s4[q], carry, c4[q] * h4[q]);
                    }
#pragma unroll
                    for (int q = 0; q < 4; ++q) hcol[i + q] = o4[q];
                }
                for (; i < j; ++i) {
                    const double hn1 = hcol[i + 1];
                    const double p = cs[i] * hn1, q = sn[i] * hn1;
                    hcol[i] = fma(cs[i], carry, q);
                    carry = fma(-sn[i], carry, p);
                }
                hcol[j] = carry;
                const double d = hypot(hcol[j], hcol[j + 1]);
                if (d == 0.0) { cs[j] = 1.0; sn[j] = 0.0; }
                else { cs[j] = hcol[j] / d; sn[j] = hcol[j + 1] / d; }
                hcol[j] = d;
                hcol[j + 1] = 0.0;
                g[j + 1] = -sn[j] * g[j];
                g[j] = cs[j] * g[j];
            }
            __syncthreads();
            PT(14)
            if (blockIdx.x == 0)
                for (int i = threadIdx.x; i <= j; i += blockDim.x) a.R[(size_t)j * (m + 1) + i] = hcol[i];
            ++iters;
            k = j + 1;
            if (a.res_hist && blockIdx.x == 0 && threadIdx.x == 0) a.res_hist[iters] = fabs(g[j + 1]) / bn;
            conv = (fabs(g[j + 1]) <= thresh) || (hn == 0.0);
            if (hn == 0.0 && !(fabs(g[j + 1]) <= thresh)) status = 2;
            __syncthreads();
            PT(4)
            if (conv || iters >= a.max_iters) break;
        }
#ifdef BIE_PHASE_TIMING
        if (threadIdx.x == 0 && blockIdx.x == 0 && MODE == 1) {
            printf("pair-loop us per step by CTA:");
            for (int c = 0; c < (int)gridDim.x; ++c) printf(" %.0f", g_pair[c] * 1e-3 / k);
            printf("\ngather us per step by CTA:");
            for (int c = 0; c < (int)gridDim.x; ++c) printf(" %.1f", g_gath[c] * 1e-3 / k);
            printf("\n");
        }
        if (threadIdx.x == 0 && pt_slot() >= 0 && !BIE_PT_PAIR_ONLY) {
            const unsigned long long* q = g_pt[pt_slot()];
            printf("cta %3d, cycle of %d steps, us per step: [operator: tables/x %.1f | pair loops or GEMV %.1f | barrier %.1f | gather %.1f | rest %.1f] "
                   "dots1 + barrier1 %.1f | reduce + w1 + tables + dots2 %.1f | barrier2 %.1f | tail %.1f (reduce2 %.1f, combine2 %.1f, v/hcol %.1f, Hf/c %.1f, Givens %.1f) | loop %.1f\n", (int)blockIdx.x, k,
                   q[6] * 1e-3 / k, q[7] * 1e-3 / k, q[8] * 1e-3 / k, q[9] * 1e-3 / k, q[0] * 1e-3 / k, q[1] * 1e-3 / k, q[2] * 1e-3 / k,
                   q[3] * 1e-3 / k, q[4] * 1e-3 / k, q[10] * 1e-3 / k, q[11] * 1e-3 / k, q[12] * 1e-3 / k, q[13] * 1e-3 / k, q[14] * 1e-3 / k, q[5] * 1e-3 / k);
        }
#endif
        // ---- a9: y = R^{-1} g (CTA 0), x += V y ---------------------------------------------------
        if (blockIdx.x == 0) {
            __syncthreads();
            // R lives in global memory (this CTA wrote it); a back-substitution that reads it from there waits one L2 round trip per
            // unknown (0.8 us each: 80 us for a full cycle of 100).  Staged into shared memory first -- the operator's scratch or the
            // slot of x, both idle here -- when the packed triangle fits.
            double* Rst = (MODE == 0) ? xs : gpart;
            const int cap = (MODE == 0) ? (XS ? n : 0) : a.scratch_doubles;
            const bool staged = (k * (k + 1) / 2 <= cap);
            if (staged) {
                for (int q = threadIdx.x >> 5; q < k; q += (int)(blockDim.x >> 5))
                    for (int i = threadIdx.x & 31; i <= q; i += 32) Rst[q * (q + 1) / 2 + i] = __ldcg(a.R + (size_t)q * (m + 1) + i);
                __syncthreads();
            }
            if (threadIdx.x < 32) {
                const int lane = threadIdx.x;
                for (int i = k - 1; i >= 0; --i) {
                    double s = 0.0;
                    if (staged) for (int c = i + 1 + lane; c < k; c += 32) s = fma(Rst[c * (c + 1) / 2 + i], hloc[c], s);
                    else for (int c = i + 1 + lane; c < k; c += 32) s = fma(a.R[(size_t)c * (m + 1) + i], hloc[c], s);
                    s = bie_warp_sum(s);
                    if (lane == 0) hloc[i] = (g[i] - s) / (staged ? Rst[i * (i + 1) / 2 + i] : a.R[(size_t)i * (m + 1) + i]);
                    __syncwarp();
                }
                for (int i = lane; i < k; i += 32) a.yv[i] = hloc[i];
            }
        }
        grid_barrier(a.sync, target);
        for (int i = threadIdx.x; i < k; i += blockDim.x) hloc[i] = __ldcg(a.yv + i);
        __syncthreads();
        basis_combine(B, rows, k, hloc, red2);
        for (int r = threadIdx.x; r < rows; r += blockDim.x) a.x[r0 + r] += red2[r];
        grid_barrier(a.sync, target);  // x complete (next residual / final residual read all of it)
        if (conv) break;
        if (iters >= a.max_iters) { status = BIE_MAX_ITERS; break; }
    }

    // ---- a10: outputs; true residual ||b - A x|| / ||b|| (reported only) -----------------------------
    double relres = 0.0;
    if (a.relres_out && bn != 0.0) {
        cta_apply<STREAM, XS, MODE>(a, r0, r1, a.x, 1.0, xs, gpart, ring, y_local, false, red, target, sb_sel);
        p = 0.0;
        for (int r = threadIdx.x; r < rows; r += blockDim.x) {
            const double v = a.b[r0 + r] - y_local[r];
            p = fma(v, v, p);
        }
        p = block_sum(p, red);
        if (threadIdx.x == 0) part1[blockIdx.x] = p;
        grid_barrier(a.sync, target);
        relres = sqrt(warp_sum_partials(part1, G)) / bn;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        if (a.iters_out) *a.iters_out = iters;
        if (a.relres_out) *a.relres_out = relres;
        if (a.status_out) *a.status_out = status;
    }
}

// ---------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------
static inline size_t al256(size_t b) { return (b + 255) & ~(size_t)255; }

struct GmresPlan {
    int G, rows_per_cta, chunk, nld, VS, scratch_doubles, brows;
    bool xs, stream;
    size_t smem;
    size_t offV, offW, offP, offR, offY, offD, offS, total;
};

// workspace layout: Krylov basis, wbuf, per-CTA partials, R, y, the stored block's product (hybrid), and the grid-barrier
// counter of the call
static void gmres_ws_layout(int n, int m, int sm_bound, GmresPlan* pl)
{
    pl->nld = (n + 1) & ~1;
    size_t o = 0;
    pl->offV = o; o += al256(sizeof(double) * (size_t)(m + 1) * pl->nld);
    pl->offW = o; o += al256(sizeof(double) * (size_t)pl->nld);
    pl->offP = o; o += al256(sizeof(double) * 3 * (size_t)(m + 2) * sm_bound);
    pl->offR = o; o += al256(sizeof(double) * (size_t)m * (m + 1));
    pl->offY = o; o += al256(sizeof(double) * (size_t)m);
    pl->offD = o; o += al256(sizeof(double) * (size_t)pl->nld);
    pl->offS = o; o += 256;
    pl->total = o;
}

static void gmres_grid(int n, int sm_count, GmresPlan* pl)
{
    // one CTA per SM whatever n is: fewer CTAs do not make the small solves faster (measured at n = 640 / 2048 / 4608 with
    // 16 ... 148 CTAs: 17.4 ... 15.9, 20.8 ... 19.0, 82 ... 35 us per iteration) -- the step is a chain of L2 round trips and
    // block barriers, not a function of the number of barrier participants
    pl->rows_per_cta = (n + sm_count - 1) / sm_count;
    pl->G = (n + pl->rows_per_cta - 1) / pl->rows_per_cta;
}

// mode: 0 stored matrix, 1 matrix-free, 2 hybrid (leading nd x nd block stored).  gmres_grid() has been called.
static int gmres_plan(int n, int restart, int sm_count, int max_smem, int l2_bytes, long long lda, int mode, int nd,
                      bool vortex, bool sym, GmresPlan* pl)
{
    const int m = restart;
    const bool free_op = (mode != 0);
    pl->brows = 0;
    if (mode == 2) {
        // every CTA streams the same number of rows of the stored block (a multiple of RING_ROWS), whoever owns them
        pl->brows = ((nd + pl->G - 1) / pl->G + RING_ROWS - 1) / RING_ROWS * RING_ROWS;
        pl->chunk = ring_chunk(pl->brows, nd, GM_WARPS - 1);
    } else {
        pl->chunk = gemv_chunk(pl->rows_per_cta, n, GM_WARPS);
    }
    pl->scratch_doubles = free_op ? free_scratch_doubles(vortex, sym) : 0;
    const int rows2 = (pl->rows_per_cta + 1) & ~1;
    size_t base = (size_t)gm_head_doubles(m, rows2, free_op);
    if (free_op) base += (size_t)pl->scratch_doubles;
    if (mode == 0) base += (size_t)((gemv_part_doubles(pl->rows_per_cta, n, pl->chunk) + 1) & ~1);
    if (mode == 2) base += (size_t)ring_part_doubles(pl->brows, nd, pl->chunk) + (size_t)ring_doubles(pl->chunk);
    base *= sizeof(double);
    base += sizeof(double) * ((size_t)GM_THREADS + rows2);  // red2
    pl->xs = mode == 0 && base + sizeof(double) * ((size_t)n + 2) <= (size_t)max_smem;
    pl->smem = base + (pl->xs ? sizeof(double) * ((size_t)n + 2) : 0);
    if (pl->smem > (size_t)max_smem) return BIE_ERR_ARG;
    // the rest of the shared memory holds this CTA's rows of as many Krylov vectors as fit
    // (dense operator: the streaming loads of A need the L1 as their landing buffer, 16 warps x 4 KB in flight,
    // so the shared-memory carve-out stops at 164 KB; measured: 408 us per step with 227 KB against 338 us.
    // The hybrid operator's block arrives by bulk copies into shared memory and needs no L1.)
    size_t cap = mode != 0 ? (size_t)max_smem : (size_t)(163 * 1024 < max_smem ? 163 * 1024 : max_smem);
#ifdef BIE_PHASE_TIMING
    cap -= 1024;   // the developer build has a few static shared variables
#endif
    pl->VS = pl->smem < cap ? (int)((cap - pl->smem) / (sizeof(double) * rows2)) : 0;
    if (pl->VS > m + 1) pl->VS = m + 1;
    pl->smem += sizeof(double) * (size_t)pl->VS * rows2;
    pl->stream = mode != 1 && (double)(mode == 2 ? nd : n) * (double)(mode == 2 ? nd : lda) * 8.0 > 0.6 * (double)l2_bytes;
    gmres_ws_layout(n, m, sm_count, pl);
    return BIE_OK;
}

size_t bie_gmres_ws_bytes(int n, int restart)
{
    if (n < 1 || restart < 1) return 0;
    if (restart > n) restart = n;
    GmresPlan pl;
    gmres_ws_layout(n, restart, 256, &pl);   // the layout depends on the device only through the SM count (<= 256)
    return pl.total + 256;                   // + alignment slack
}

template <bool STREAM, bool XS, int MODE>
static int launch_gmres(bie_ctx* ctx, const GmresArgs& a, const GmresPlan& pl, cudaStream_t st)
{
    auto k = bie_gmres_kernel<STREAM, XS, MODE>;
    const int rc = bie_grant_smem(ctx, (MODE == 0 ? (STREAM ? 2 : 0) + (XS ? 1 : 0) : (MODE == 1 ? 4 : 5 + (STREAM ? 1 : 0))), k, pl.smem);
    if (rc != BIE_OK) return rc;
    void* params[] = {(void*)&a};
    BIE_CUDA(cudaLaunchCooperativeKernel((const void*)k, dim3(pl.G), dim3(GM_THREADS), params, pl.smem, st));
    return BIE_OK;
}

// nd == 0: stored matrix (A != NULL) or matrix-free (A == NULL); 0 < nd < n (even): hybrid, A holds the columns [0, nd)
int bie_launch_gmres(bie_ctx* ctx, int n, const double* A, int64_t lda, int nd, const double* rhs, double tol,
                     int restart, int max_iters, double* x, int32_t* iters_out, double* relres_out,
                     int32_t* status_out, double* res_hist, void* ws, size_t ws_bytes, cudaStream_t st)
{
    if (!ctx || !rhs || !x || !ws) return BIE_ERR_NULL;
    if (n < 1 || restart < 1 || max_iters < 0 || !(tol >= 0.0)) return BIE_ERR_ARG;
    if (nd < 0 || nd >= n || (nd & 1) || (nd > 0 && !A)) return nd > 0 && !A ? BIE_ERR_NULL : BIE_ERR_ARG;
    const int mode = nd > 0 ? 2 : (A == nullptr ? 1 : 0);
    const bool free_op = (mode != 0);
    if (free_op && (!ctx->have_geom || ctx->n != n)) return BIE_ERR_GEOMETRY;
    if (mode == 0 && (lda < n || (lda & 1))) return BIE_ERR_LAYOUT;     // hybrid: A is in the block format, lda is not used
    if (mode != 1 && (((uintptr_t)A) & 15u)) return BIE_ERR_LAYOUT;
    if ((((uintptr_t)rhs) | ((uintptr_t)x)) & 15u) return BIE_ERR_LAYOUT;
    if (!ctx->coop_ok) return BIE_ERR_DEVICE;
    if (ctx->sm_count > 256) return BIE_ERR_DEVICE;
    if (restart > n) restart = n;  // the Krylov space cannot exceed n
    GmresPlan pl;
    gmres_grid(n, ctx->sm_count, &pl);
    GmresArgs a;
    memset(&a.nt, 0, sizeof(a.nt)); memset(&a.ct, 0, sizeof(a.ct)); memset(&a.fp, 0, sizeof(a.fp));
    int rc;
    if (free_op) {
        a.nt = bie_node_table(ctx); a.ct = ctx->comps;
        rc = bie_ensure_near(ctx, st);
        if (rc != BIE_OK) return rc;
        rc = bie_free_plan(ctx, pl.G, nd, &a.fp, st);     // decides one-directional / symmetric loops; checks nd
        if (rc != BIE_OK) return rc;
    }
    rc = gmres_plan(n, restart, ctx->sm_count, ctx->max_smem_optin, ctx->l2_bytes, free_op ? n : lda, mode, nd,
                    a.fp.vortex != 0, a.fp.sym != 0, &pl);
    if (rc != BIE_OK) return rc;
    // align the caller's workspace to 256 bytes
    uintptr_t base = ((uintptr_t)ws + 255) & ~(uintptr_t)255;
    if (base - (uintptr_t)ws + pl.total > ws_bytes) return BIE_ERR_WORKSPACE;
    a.A = A; a.lda = lda; a.n = n; a.b = rhs; a.tol = tol; a.m = restart; a.max_iters = max_iters;
    a.x = x; a.iters_out = iters_out; a.relres_out = relres_out; a.status_out = status_out; a.res_hist = res_hist;
    a.V = (double*)(base + pl.offV);
    a.wbuf = (double*)(base + pl.offW);
    a.part = (double*)(base + pl.offP);
    a.R = (double*)(base + pl.offR);
    a.yv = (double*)(base + pl.offY);
    a.yd = (double*)(base + pl.offD);
    a.sync = (unsigned int*)(base + pl.offS);     // per call: two solves of one ctx never share a barrier counter
    a.nld = pl.nld; a.rows_per_cta = pl.rows_per_cta; a.chunk = pl.chunk; a.VS = pl.VS;
    a.nd = nd; a.nwf = ctx->hybrid_free_warps; a.poll_tiles = ctx->hybrid_poll_tiles; a.scratch_doubles = pl.scratch_doubles; a.brows = pl.brows;
    a.res_pairs = (mode == 0 && pl.stream)
        ? bie_gemv_resident_pairs(ctx->l2_bytes, n, (long long)lda, pl.rows_per_cta, sizeof(double) * (size_t)(restart + 2) * pl.nld) : 0;
    BIE_CUDA(cudaMemsetAsync(a.sync, 0, sizeof(unsigned int), st));
    if (mode == 0) {
        // small stored-matrix systems: one thread-block cluster, distributed shared memory instead of grid barriers and L2
        // (bie_gmres_cluster.cu); same workspace layout
        rc = bie_launch_gmres_cluster(ctx, n, A, lda, rhs, tol, restart, max_iters, x, iters_out, relres_out, status_out, res_hist,
                                      a.V, pl.nld, a.R, st);
        if (rc != BIE_CLUSTER_NOT_TAKEN) return rc;
    }
    if (mode == 1) return launch_gmres<false, false, 1>(ctx, a, pl, st);
    if (mode == 2) return pl.stream ? launch_gmres<true, true, 2>(ctx, a, pl, st) : launch_gmres<false, true, 2>(ctx, a, pl, st);
    if (pl.stream) return pl.xs ? launch_gmres<true, true, 0>(ctx, a, pl, st) : launch_gmres<true, false, 0>(ctx, a, pl, st);
    return pl.xs ? launch_gmres<false, true, 0>(ctx, a, pl, st) : launch_gmres<false, false, 0>(ctx, a, pl, st);
}
