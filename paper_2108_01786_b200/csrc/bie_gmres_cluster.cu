// bie_gmres_cluster.cu -- SURVEY 8(a) rows a5-a10 for SMALL systems (n <= BIE_CLUSTER_MAX_N): the restarted GMRES(m) of
// bie_gmres.cu (Saad & Schultz, ref. [38] at PAPER.md:L855; stopping rule PAPER.md:L869) on ONE thread-block cluster.
//
// Why: with a stored matrix of a few MB the grid-wide kernel of bie_gmres.cu is a chain of L2 round trips -- two grid
// barriers through a global counter (1.5-2 us each) and two reductions of per-CTA partials read back from L2 (1.4-2.3 us
// each) per Arnoldi step: 13.5 us per step at n = 640 against 0.5 us for the GEMV itself.  A cluster of 16 (or 8) CTAs has
// what such a solve needs ON the chip: distributed shared memory instead of L2 for everything that crosses CTAs.
//   - CTA c owns a contiguous block of rows of A, of every Krylov vector and of x.  Its rows of A sit in its shared
//     memory for the whole solve (at n = 640: 36 of its 40 rows; the others stream from L2, split over all warps and
//     issued before the shared-memory rows of every GEMV).
//   - exchanges: a CTA sends its rows of the next Krylov vector (or its partial dot products) into the shared memory
//     of EVERY CTA of the cluster with st.async, whose completion the hardware counts in bytes on an mbarrier of the
//     RECEIVER (mbarrier::complete_tx); the receiver states how many bytes the exchange brings (arrive.expect_tx) and
//     waits for the phase.  No cluster-wide barrier and no fence per exchange (the first version used remote stores +
//     barrier.cluster: its release/acquire fences were 2.3 of 15 stall cycles per issue, profiles/r02b_cluster.md).  Every CTA
//     adds the partials by the same xor-shuffle tree -- all CTAs hold bit-identical coefficients, Givens rotations and
//     residuals and take the same branches without further communication.
//   - Arnoldi step j: y = A v_j (shared memory);  s = V_j^T y (exchange 1);  w1 = y - V_j s;
//     h2 = V_j^T w1 and ||w1||^2 (exchange 2);  hn^2 = ||w1||^2 - ||h2||^2 (Pythagoras, as bie_gmres.cu;
//     explicit norm with one more exchange when h2 is not small);  v_{j+1} = (w1 - V_j h2)/hn -> all CTAs (exchange 3, which
//     lands while one thread runs the Givens sweep).  Classical Gram-Schmidt twice (CGS2), h = s + h2, Givens and the
//     recurrence residual as in bie_gmres.cu (a8), back-substitution by CTA 0 at the end of a cycle (a9), true residual at
//     the end (a10).
// Buffer reuse needs no extra synchronisation: the partial buffers alternate between two copies (each with its own
// mbarrier), and a CTA can send exchange k + 2 only after it has received everyone's exchange k + 1, which every CTA sends
// after it has consumed exchange k.  A variant with the whole basis REPLICATED in every CTA of the full grid (one grid
// barrier per step, Gram-Schmidt local and redundant) was built too and is slower (14-20 us per step at n = 640: four passes
// over the basis per step through one SM's shared-memory port): DESIGN.md section 7d.
#include <cooperative_groups.h>
#include "bie_common.cuh"

namespace cg = cooperative_groups;


#define CL_THREADS 512
#define CL_WARPS (CL_THREADS / 32)

struct ClusterArgs {
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
    double* res_hist;
    double* Vg;        // global spill of the basis, [(m+1)][nld] (vectors VS.. only)
    int nld;
    double* R;         // [m][m+1], column j at R + j (m + 1); CTA 0 only
    int rows_per_cta;
    int rows_smem;     // rows of A per CTA kept in shared memory
    int VS;            // Krylov vectors 0..VS-1 keep this CTA's rows in shared memory
    int mp;            // stride of one CTA's slot in the partial buffers, >= m + 2
};

// shared-memory plan (doubles), the same on host and device
struct ClusterSmem {
    int xs, y, w, xl, dl, hloc, hcol, cs, sn, g, red, P, Vs, As, total;
};

__host__ __device__ inline ClusterSmem cluster_smem(int n, int m, int rows_per_cta, int mp, int CS, int VS, int rows_smem)
{
    const int n2 = (n + 1) & ~1, rows2 = (rows_per_cta + 1) & ~1, m2 = (m + 3) & ~1;
    ClusterSmem s;
    int o = 0;
    s.xs = o; o += n2;              // the operator's input vector, complete (written by all CTAs)
    s.y = o; o += rows2;            // result of the operator on this CTA's rows
    s.w = o; o += rows2;            // the vector being orthogonalised
    s.xl = o; o += rows2;           // this CTA's rows of x
    s.dl = o; o += m2;              // local dot products
    s.hloc = o; o += m2;            // reduced coefficients of the current pass
    s.hcol = o; o += m2;            // column j of H
    s.cs = o; o += m2;
    s.sn = o; o += m2;
    s.g = o; o += m2;
    s.red = o; o += 40;
    s.P = o; o += 2 * CS * mp;      // all-gathered partials, two copies
    s.Vs = o; o += VS * rows2;
    s.As = o; o += rows_smem * n2;
    s.total = o;
    return s;
}

__device__ __forceinline__ double cl_block_sum(double v, double* red)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    v = bie_warp_sum(v);
    __syncthreads();
    if (lane == 0) red[warp] = v;
    __syncthreads();
    if (warp == 0) {
        double s = (lane < CL_WARPS) ? red[lane] : 0.0;
        s = bie_warp_sum(s);
        if (lane == 0) red[32] = s;
    }
    __syncthreads();
    return red[32];
}

// ---- exchange primitives: st.async into a peer's shared memory, completion counted in bytes on the PEER's mbarrier ----
__device__ __forceinline__ uint32_t cl_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t cl_mapa(uint32_t addr, int rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
__device__ __forceinline__ void cl_st_async(uint32_t remote_addr, double v, uint32_t remote_mbar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b64 [%0], %1, [%2];"
                 :: "r"(remote_addr), "l"(__double_as_longlong(v)), "r"(remote_mbar) : "memory");
}
__device__ __forceinline__ void cl_mbar_init(uint32_t mb, int count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(mb), "r"(count) : "memory"); }
__device__ __forceinline__ void cl_mbar_expect(uint32_t mb, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(mb), "r"(bytes) : "memory");
}
// all bytes of the phase with this parity have landed (and are visible: acquire at cluster scope)
__device__ __forceinline__ void cl_mbar_wait(uint32_t mb, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(mb), "r"(parity) : "memory");
    } while (!done);
}

struct ClusterCtx {
    cg::cluster_group cl;
    int rank, CS;
    int r0, rows, rows2, n, n2, mp;
    double* smem;
    ClusterSmem L;
    unsigned kP;     // exchanges of partial sums so far: exchange k uses buffer and mbarrier k & 1, phase parity (k >> 1) & 1
    unsigned kX;     // all-gathers of a vector into xs so far (one mbarrier, parity kX & 1)
    uint32_t mbP, mbX, mbY;   // shared addresses of the mbarriers: partial sums [2], vector, the solution of the small least-squares problem
};

// vals[0..cnt) (shared) of every CTA -> out[i] = sum over the CTAs, in every CTA: the same fixed tree everywhere (lane q of a
// group of CS lanes holds CTA q's partial; xor-shuffle tree), so all CTAs get the same bits.  ssq != NULL: *ssq = sum of
// out[i]^2 over i < cnt - 1 (the norm of h2 in the second Gram-Schmidt pass), by warp 0 in fixed order.  Ends with __syncthreads.
__device__ __forceinline__ void cl_allreduce(ClusterCtx& c, const double* vals, int cnt, double* out, double* ssq = nullptr)
{
    const unsigned k = c.kP++;
    double* P = c.smem + c.L.P + (k & 1) * c.CS * c.mp;
    const uint32_t mb = c.mbP + 8 * (k & 1);
    const int sh = (c.CS == 16) ? 4 : 3;                      // CS is 16 or 8
    if (threadIdx.x == 0) cl_mbar_expect(mb, (uint32_t)(cnt << sh) * 8u);      // every CTA (this one too) sends cnt doubles
    const uint32_t slot = cl_smem_u32(P + c.rank * c.mp);
    for (int t = threadIdx.x; t < (cnt << sh); t += CL_THREADS) {
        const int peer = t & (c.CS - 1), i = t >> sh;
        cl_st_async(cl_mapa(slot + 8 * i, peer), vals[i], cl_mapa(mb, peer));
    }
    cl_mbar_wait(mb, (k >> 1) & 1);
    const int per = CL_THREADS >> sh;                          // values per pass of the whole CTA
    for (int i0 = 0; i0 < cnt; i0 += per) {
        const int i = i0 + (threadIdx.x >> sh), q = threadIdx.x & (c.CS - 1);
        double v = (i < cnt) ? P[q * c.mp + i] : 0.0;
        for (int o = c.CS >> 1; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (i < cnt && q == 0) out[i] = v;
    }
    __syncthreads();
    if (ssq != nullptr) {
        if (threadIdx.x < 32) {
            double ss = 0.0;
            for (int i = threadIdx.x; i < cnt - 1; i += 32) ss = fma(out[i], out[i], ss);
            ss = bie_warp_sum(ss);
            if (threadIdx.x == 0) *ssq = ss;
        }
        __syncthreads();
    }
}

// this CTA's rows of a vector (shared, v[0..rows)) -> xs of every CTA (non-blocking); cl_xs_wait() before xs is read
__device__ __forceinline__ void cl_allgather_rows(ClusterCtx& c, const double* v)
{
    const uint32_t xs0 = cl_smem_u32(c.smem + c.L.xs + c.r0);
    if (threadIdx.x == 0) cl_mbar_expect(c.mbX, (uint32_t)c.n * 8u);           // all n entries arrive, this CTA's own too
    for (int t = threadIdx.x; t < c.rows * c.CS; t += CL_THREADS) {
        const int peer = t / c.rows, i = t - peer * c.rows;
        cl_st_async(cl_mapa(xs0 + 8 * i, peer), v[i], cl_mapa(c.mbX, peer));
    }
}
__device__ __forceinline__ void cl_xs_wait(ClusterCtx& c)
{
    cl_mbar_wait(c.mbX, c.kX & 1);
    ++c.kX;
}

// y[r] = A[r0 + r, :] xs for this CTA's rows.  Rows in shared memory: one warp per row.  The rows that did not fit stream
// from L2: every warp takes a sixteenth of each of them (at most 32 pairs of columns: n <= 1024), issues its loads for a batch
// of CL_GB rows BEFORE the shared-memory rows and multiplies afterwards, so the L2 latency hides behind those; the warps'
// sums of a row are added in fixed order.  gpart: shared, [CL_GB][CL_WARPS].  Ends with __syncthreads.
#define CL_GB 4
#define CL_RW 3
__device__ __forceinline__ void cl_gemv(const ClusterCtx& c, const ClusterArgs& a, double* y, double* gpart)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const double* xs = c.smem + c.L.xs;
    const double* As = c.smem + c.L.As;
    const int npair = c.n >> 1;
    const int nsm = min(c.rows, a.rows_smem), ng = c.rows - nsm;
    const int chunk = (npair + CL_WARPS - 1) / CL_WARPS;             // pairs of columns per warp and streamed row, <= 32
    const int pg = warp * chunk + lane;                                // this lane's pair of a streamed row
    const bool have = (lane < chunk) && (pg < npair);
    double2 gv[CL_GB];
    auto issue = [&](int g0) {
#pragma unroll
        for (int q = 0; q < CL_GB; ++q) {
            gv[q] = make_double2(0.0, 0.0);
            if (g0 + q < ng && have)
                gv[q] = __ldcg(reinterpret_cast<const double2*>(a.A + (size_t)(c.r0 + nsm + g0 + q) * a.lda) + pg);
        }
    };
    auto consume = [&](int g0) {
        const double2 xv = have ? reinterpret_cast<const double2*>(xs)[pg] : make_double2(0.0, 0.0);
#pragma unroll
        for (int q = 0; q < CL_GB; ++q) {
            double s = fma(gv[q].x, xv.x, gv[q].y * xv.y);
            if ((c.n & 1) && warp == CL_WARPS - 1 && lane == 0 && g0 + q < ng)      // odd n: the last column
                s = fma(__ldcg(a.A + (size_t)(c.r0 + nsm + g0 + q) * a.lda + c.n - 1), xs[c.n - 1], s);
            s = bie_warp_sum(s);
            if (lane == 0) gpart[q * CL_WARPS + warp] = s;
        }
    };
    if (ng > 0) issue(0);
    // up to CL_RW rows of a warp together: one load of the x pair serves them all (the shared-memory bandwidth, 128 B per
    // clock, is what bounds this loop), and their lane reductions overlap
    for (int rb = warp; rb < nsm; rb += CL_RW * CL_WARPS) {
        double s0[CL_RW], s1[CL_RW];
        const double2* row[CL_RW];
#pragma unroll
        for (int q = 0; q < CL_RW; ++q) {
            s0[q] = 0.0; s1[q] = 0.0;
            row[q] = reinterpret_cast<const double2*>(As + (size_t)min(rb + q * CL_WARPS, nsm - 1) * c.n2);
        }
        for (int p = lane; p < npair; p += 32) {
            const double2 xv = reinterpret_cast<const double2*>(xs)[p];
#pragma unroll
            for (int q = 0; q < CL_RW; ++q) {
                const double2 av = row[q][p];
                s0[q] = fma(av.x, xv.x, s0[q]); s1[q] = fma(av.y, xv.y, s1[q]);
            }
        }
#pragma unroll
        for (int q = 0; q < CL_RW; ++q) {
            const int r = rb + q * CL_WARPS;
            if ((c.n & 1) && lane == 0 && r < nsm) s0[q] = fma(As[(size_t)r * c.n2 + c.n - 1], xs[c.n - 1], s0[q]);
            const double t = bie_warp_sum(s0[q] + s1[q]);
            if (lane == 0 && r < nsm) y[r] = t;
        }
    }
    for (int g0 = 0; g0 < ng; g0 += CL_GB) {
        consume(g0);
        __syncthreads();
        if (threadIdx.x < CL_GB * CL_WARPS) {           // the warps' sums of a row: 16 lanes, the same xor tree everywhere
            double t = gpart[threadIdx.x];
            for (int o = CL_WARPS >> 1; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
            const int q = threadIdx.x / CL_WARPS;
            if ((threadIdx.x & (CL_WARPS - 1)) == 0 && g0 + q < ng) y[nsm + g0 + q] = t;
        }
        if (g0 + CL_GB < ng) { __syncthreads(); issue(g0 + CL_GB); }
    }
    __syncthreads();
}

// this CTA's rows of Krylov vector i
__device__ __forceinline__ double* cl_vec(const ClusterCtx& c, const ClusterArgs& a, int i)
{
    return (i < a.VS) ? c.smem + c.L.Vs + (size_t)i * c.rows2 : a.Vg + (size_t)i * a.nld + c.r0;
}

// dl[i] = <v_i, w>_rows for i < cnt; with_norm: dl[cnt] = ||w||_rows^2.  Ends with __syncthreads.
__device__ __forceinline__ void cl_local_dots(const ClusterCtx& c, const ClusterArgs& a, int cnt, const double* w, double* dl, bool with_norm)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int tot = cnt + (with_norm ? 1 : 0);
    for (int i = warp; i < tot; i += CL_WARPS) {
        const double* vi = (i == cnt) ? w : cl_vec(c, a, i);
        double s = 0.0;
        for (int r = lane; r < c.rows; r += 32) s = fma(vi[r], w[r], s);
        s = bie_warp_sum(s);
        if (lane == 0) dl[i] = s;
    }
    __syncthreads();
}

// w[r] -= sum_{i < cnt} coef[i] v_i[r] on this CTA's rows: groups of 32 threads take every (CL_THREADS/32)-th vector... the
// rows are few (n / cluster size), so thread (r, g) sums the vectors i = g, g + G, ... and the G group sums are added in
// fixed order.  scratch: shared, >= CL_THREADS doubles.  Ends with __syncthreads.
__device__ __forceinline__ void cl_subtract_combination(const ClusterCtx& c, const ClusterArgs& a, int cnt, const double* coef,
                                                        double* w, double* scratch)
{
    int rp = 1;
    while (rp < c.rows) rp <<= 1;               // rows rounded up to a power of two <= CL_THREADS (rows <= 64 by the plan)
    const int G = CL_THREADS / rp;
    const int g = threadIdx.x / rp, r = threadIdx.x - g * rp;
    double s = 0.0;
    if (r < c.rows)
        for (int i = g; i < cnt; i += G) s = fma(coef[i], cl_vec(c, a, i)[r], s);
    scratch[threadIdx.x] = s;
    __syncthreads();
    if (threadIdx.x < c.rows) {
        double t = 0.0;
        for (int q = 0; q < G; ++q) t += scratch[q * rp + threadIdx.x];
        w[threadIdx.x] -= t;
    }
    __syncthreads();
}

__global__ void __launch_bounds__(CL_THREADS, 1) bie_gmres_cluster_kernel(const ClusterArgs a)
{
    extern __shared__ __align__(16) double smem[];
    ClusterCtx c{cg::this_cluster()};
    c.rank = (int)c.cl.block_rank(); c.CS = (int)c.cl.num_blocks();
    c.n = a.n; c.n2 = (a.n + 1) & ~1; c.mp = a.mp;
    c.r0 = min(c.rank * a.rows_per_cta, a.n);
    c.rows = min(c.r0 + a.rows_per_cta, a.n) - c.r0;      // may be 0 for the last CTAs of a tiny system
    c.rows2 = (a.rows_per_cta + 1) & ~1;
    c.smem = smem; c.kP = 0; c.kX = 0;
    __shared__ __align__(8) unsigned long long mbar[4];
    c.mbP = cl_smem_u32(&mbar[0]); c.mbX = cl_smem_u32(&mbar[2]); c.mbY = cl_smem_u32(&mbar[3]);
    if (threadIdx.x == 0) {
        for (int q = 0; q < 4; ++q) cl_mbar_init(c.mbP + 8 * q, 1);      // one arrival per phase: the thread that states the expected bytes
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    unsigned kY = 0;
    c.L = cluster_smem(a.n, a.m, a.rows_per_cta, a.mp, c.CS, a.VS, a.rows_smem);
    const int m = a.m, rows = c.rows, r0 = c.r0;
    double* y = smem + c.L.y;  double* w = smem + c.L.w;  double* xl = smem + c.L.xl;
    double* dl = smem + c.L.dl;  double* hloc = smem + c.L.hloc;  double* hcol = smem + c.L.hcol;
    double* cs = smem + c.L.cs;  double* sn = smem + c.L.sn;  double* g = smem + c.L.g;  double* red = smem + c.L.red;
    __shared__ double comb[CL_THREADS];

    // ---- this CTA's rows of A -> shared memory ----------------------------------------------------------------
    {
        const int nsm = min(rows, a.rows_smem), npair = a.n >> 1;
        double* As = smem + c.L.As;
        for (int r = threadIdx.x >> 5; r < nsm; r += CL_WARPS) {
            const double* grow = a.A + (size_t)(r0 + r) * a.lda;
            for (int p = threadIdx.x & 31; p < npair; p += 32)
                reinterpret_cast<double2*>(As + (size_t)r * c.n2)[p] = __ldcs(reinterpret_cast<const double2*>(grow) + p);
            if ((a.n & 1) && (threadIdx.x & 31) == 0) As[(size_t)r * c.n2 + a.n - 1] = grow[a.n - 1];
        }
    }
    __syncthreads();
    // ---- a5: ||b||, x = 0 ---------------------------------------------------------------------------------------
    double p = 0.0;
    for (int r = threadIdx.x; r < rows; r += CL_THREADS) {
        const double v = a.b[r0 + r];
        p = fma(v, v, p);
        xl[r] = 0.0;
    }
    p = cl_block_sum(p, red);
    if (threadIdx.x == 0) dl[0] = p;
    __syncthreads();
    c.cl.sync();                                   // every CTA of the cluster is running: remote shared memory may be written
    cl_allreduce(c, dl, 1, hloc);
    const double bn = sqrt(hloc[0]);
    const double thresh = a.tol * bn;
    __syncthreads();

    int iters = 0, status = 0;
    bool done = (bn == 0.0), first = true;
    if (a.res_hist && c.rank == 0 && threadIdx.x == 0) a.res_hist[0] = 1.0;
    while (!done) {
        // ---- cycle start: r = b - A x -----------------------------------------------------------------------------
        if (first) {
            for (int r = threadIdx.x; r < rows; r += CL_THREADS) w[r] = a.b[r0 + r];
            first = false;
            __syncthreads();
        } else {
            cl_allgather_rows(c, xl);
            cl_xs_wait(c);
            cl_gemv(c, a, y, comb);
            for (int r = threadIdx.x; r < rows; r += CL_THREADS) w[r] = a.b[r0 + r] - y[r];
            __syncthreads();
        }
        p = 0.0;
        for (int r = threadIdx.x; r < rows; r += CL_THREADS) p = fma(w[r], w[r], p);
        p = cl_block_sum(p, red);
        if (threadIdx.x == 0) dl[0] = p;
        __syncthreads();
        cl_allreduce(c, dl, 1, hloc);
        const double beta = sqrt(hloc[0]);
        __syncthreads();
        if (beta <= thresh) break;                         // converged (status 0)
        if (iters >= a.max_iters) { status = BIE_MAX_ITERS; break; }
        {
            const double inv = 1.0 / beta;
            double* v0 = cl_vec(c, a, 0);
            for (int r = threadIdx.x; r < rows; r += CL_THREADS) { const double v = w[r] * inv; v0[r] = v; w[r] = v; }
            __syncthreads();
            cl_allgather_rows(c, w);
            cl_xs_wait(c);
        }
        if (threadIdx.x == 0) g[0] = beta;
        __syncthreads();

        // ---- Arnoldi steps ------------------------------------------------------------------------------------------
        int k = 0;
        bool conv = false;
        for (int j = 0; j < m; ++j) {
            cl_gemv(c, a, y, comb);                                              // a6: y = A v_j
            // a7, first pass: s = V_j^T y, w1 = y - V_j s
            cl_local_dots(c, a, j + 1, y, dl, false);
            cl_allreduce(c, dl, j + 1, hloc);
            for (int i = threadIdx.x; i <= j; i += CL_THREADS) hcol[i] = hloc[i];
            for (int r = threadIdx.x; r < rows; r += CL_THREADS) w[r] = y[r];
            __syncthreads();
            cl_subtract_combination(c, a, j + 1, hloc, w, comb);
            // second pass: h2 = V_j^T w1 and ||w1||^2 in one reduction
            cl_local_dots(c, a, j + 1, w, dl, true);
            cl_allreduce(c, dl, j + 2, hloc, red + 34);                   // red[34] = ||h2||^2
            const double nu = hloc[j + 1], ss = red[34];
            cl_subtract_combination(c, a, j + 1, hloc, w, comb);         // w2 = w1 - V_j h2
            double hn;
            if (ss <= 0.01 * nu) {                                         // identical in every CTA (same bits)
                hn = sqrt(nu - ss);                                        // Pythagoras: no cancellation, ss << nu
            } else {                                                       // breakdown region: explicit norm
                p = 0.0;
                for (int r = threadIdx.x; r < rows; r += CL_THREADS) p = fma(w[r], w[r], p);
                p = cl_block_sum(p, red);
                if (threadIdx.x == 0) dl[0] = p;
                __syncthreads();
                cl_allreduce(c, dl, 1, red + 36);
                hn = sqrt(red[36]);
            }
            for (int i = threadIdx.x; i <= j; i += CL_THREADS) hcol[i] += hloc[i];
            {
                const double inv = (hn != 0.0) ? 1.0 / hn : 0.0;
                double* vn = cl_vec(c, a, j + 1);
                for (int r = threadIdx.x; r < rows; r += CL_THREADS) { const double v = w[r] * inv; vn[r] = v; w[r] = v; }
            }
            __syncthreads();
            cl_allgather_rows(c, w);                                       // v_{j+1} -> xs of every CTA; the Givens sweep runs while it lands
            // a8: Givens rotations on column j, new rotation, recurrence residual (one thread, the same bits in every CTA)
            if (threadIdx.x == CL_THREADS - 1) {
                hcol[j + 1] = hn;
                for (int i = 0; i < j; ++i) {
                    const double t0 = cs[i] * hcol[i] + sn[i] * hcol[i + 1];
                    const double t1 = -sn[i] * hcol[i] + cs[i] * hcol[i + 1];
                    hcol[i] = t0;
                    hcol[i + 1] = t1;
                }
                const double d = hypot(hcol[j], hcol[j + 1]);
                if (d == 0.0) { cs[j] = 1.0; sn[j] = 0.0; }
                else { cs[j] = hcol[j] / d; sn[j] = hcol[j + 1] / d; }
                hcol[j] = d;
                hcol[j + 1] = 0.0;
                g[j + 1] = -sn[j] * g[j];
                g[j] = cs[j] * g[j];
            }
            cl_xs_wait(c);
            __syncthreads();
            if (c.rank == 0)
                for (int i = threadIdx.x; i <= j; i += CL_THREADS) a.R[(size_t)j * (m + 1) + i] = hcol[i];
            ++iters;
            k = j + 1;
            if (a.res_hist && c.rank == 0 && threadIdx.x == 0) a.res_hist[iters] = fabs(g[j + 1]) / bn;
            conv = (fabs(g[j + 1]) <= thresh) || (hn == 0.0);
            if (hn == 0.0 && !(fabs(g[j + 1]) <= thresh)) status = 2;
            __syncthreads();
            if (conv || iters >= a.max_iters) break;
        }
        // ---- a9: y = R^{-1} g (CTA 0) -> every CTA, x += V y -----------------------------------------------------------
        if (c.rank == 0) {
            __syncthreads();
            // R (global, written by this CTA) is staged into the partial buffers first -- idle here: no CTA sends partial sums before it has
            // the solution of this cycle -- so that the back-substitution does not wait one L2 round trip per unknown
            double* Rst = smem + c.L.P;
            const bool staged = (k * (k + 1) / 2 <= 2 * c.CS * c.mp);
            if (staged) {
                for (int q = threadIdx.x >> 5; q < k; q += CL_WARPS)
                    for (int i = threadIdx.x & 31; i <= q; i += 32) Rst[q * (q + 1) / 2 + i] = __ldcg(a.R + (size_t)q * (m + 1) + i);
                __syncthreads();
            }
            if (threadIdx.x < 32) {
                const int lane = threadIdx.x;
                for (int i = k - 1; i >= 0; --i) {
                    double s = 0.0;
                    if (staged) for (int q = i + 1 + lane; q < k; q += 32) s = fma(Rst[q * (q + 1) / 2 + i], hloc[q], s);
                    else for (int q = i + 1 + lane; q < k; q += 32) s = fma(a.R[(size_t)q * (m + 1) + i], hloc[q], s);
                    s = bie_warp_sum(s);
                    if (lane == 0) hloc[i] = (g[i] - s) / (staged ? Rst[i * (i + 1) / 2 + i] : a.R[(size_t)i * (m + 1) + i]);
                    __syncwarp();
                }
            }
            __syncthreads();
            for (int t = threadIdx.x; t < k * c.CS; t += CL_THREADS) {         // y -> hloc of every CTA (this one too: the same values)
                const int peer = t / k, i = t - peer * k;
                cl_st_async(cl_mapa(cl_smem_u32(hloc + i), peer), hloc[i], cl_mapa(c.mbY, peer));
            }
        }
        if (threadIdx.x == 0) cl_mbar_expect(c.mbY, (uint32_t)k * 8u);
        cl_mbar_wait(c.mbY, kY & 1);
        ++kY;
        __syncthreads();
        for (int r = threadIdx.x; r < rows; r += CL_THREADS) w[r] = -xl[r];
        __syncthreads();
        cl_subtract_combination(c, a, k, hloc, w, comb);                  // w = -(x + V y)
        for (int r = threadIdx.x; r < rows; r += CL_THREADS) xl[r] = -w[r];
        __syncthreads();
        if (conv) break;
        if (iters >= a.max_iters) { status = BIE_MAX_ITERS; break; }
    }

    // ---- a10: outputs; true residual ||b - A x|| / ||b|| (reported only) ------------------------------------------------
    for (int r = threadIdx.x; r < rows; r += CL_THREADS) a.x[r0 + r] = xl[r];
    double relres = 0.0;
    if (a.relres_out && bn != 0.0) {
        cl_allgather_rows(c, xl);
        cl_xs_wait(c);
        cl_gemv(c, a, y, comb);
        p = 0.0;
        for (int r = threadIdx.x; r < rows; r += CL_THREADS) {
            const double v = a.b[r0 + r] - y[r];
            p = fma(v, v, p);
        }
        p = cl_block_sum(p, red);
        if (threadIdx.x == 0) dl[0] = p;
        __syncthreads();
        cl_allreduce(c, dl, 1, hloc);
        relres = sqrt(hloc[0]) / bn;
    }
    if (c.rank == 0 && threadIdx.x == 0) {
        if (a.iters_out) *a.iters_out = iters;
        if (a.relres_out) *a.relres_out = relres;
        if (a.status_out) *a.status_out = status;
    }
    c.cl.sync();      // no CTA exits while another may still write into its shared memory
}

// ---------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------

// cluster size this device can co-schedule with the kernel's full shared memory: 16 (non-portable), else 8, else -1
static int cluster_probe(bie_ctx* ctx)
{
    if (ctx->cluster_size != 0) return ctx->cluster_size;
    ctx->cluster_size = -1;
    if (cudaFuncSetAttribute(bie_gmres_cluster_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, ctx->max_smem_optin - 4096 - (int)sizeof(double) * CL_THREADS) != cudaSuccess ||
        cudaFuncSetAttribute(bie_gmres_cluster_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) {
        cudaGetLastError();
        return -1;
    }
    for (int cs = 16; cs >= 8; cs >>= 1) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(cs); cfg.blockDim = dim3(CL_THREADS);
        cfg.dynamicSmemBytes = (size_t)(ctx->max_smem_optin - 4096 - (int)sizeof(double) * CL_THREADS);
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        int nclusters = 0;
        if (cudaOccupancyMaxActiveClusters(&nclusters, bie_gmres_cluster_kernel, &cfg) == cudaSuccess && nclusters >= 1) {
            ctx->cluster_size = cs;
            break;
        }
        cudaGetLastError();
    }
    return ctx->cluster_size;
}

// BIE_OK: launched.  BIE_CLUSTER_NOT_TAKEN (> 0): this solve is not for the cluster kernel, the caller goes on with the grid-wide one.
int bie_launch_gmres_cluster(bie_ctx* ctx, int n, const double* A, int64_t lda, const double* rhs, double tol, int restart,
                             int max_iters, double* x, int32_t* iters_out, double* relres_out, int32_t* status_out,
                             double* res_hist, double* Vg, int nld, double* R, cudaStream_t st)
{
    if (!ctx->small_gmres || n > BIE_CLUSTER_MAX_N) return BIE_CLUSTER_NOT_TAKEN;
    const int CS = cluster_probe(ctx);
    if (CS < 8) return BIE_CLUSTER_NOT_TAKEN;
    const int m = restart;
    ClusterArgs a;
    a.rows_per_cta = (n + CS - 1) / CS;
    if (a.rows_per_cta > 64) return BIE_CLUSTER_NOT_TAKEN;       // cl_subtract_combination: rows <= CL_THREADS / 8
    a.mp = (m + 2) | 1;            // odd: the CTAs' slots fall on different banks
    const int budget = (ctx->max_smem_optin - 4096 - (int)sizeof(double) * CL_THREADS) / (int)sizeof(double);
    const int n2 = (n + 1) & ~1, rows2 = (a.rows_per_cta + 1) & ~1;
    // the Krylov basis first (a vector outside costs four exposed L2 round trips per step, a row of A outside only its
    // bytes, which stream while the other rows are multiplied), then as many rows of A as fit
    const ClusterSmem base = cluster_smem(n, m, a.rows_per_cta, a.mp, CS, 0, 0);
    if (base.total + rows2 > budget) return BIE_CLUSTER_NOT_TAKEN;
    const int left = budget - base.total;
    a.VS = left / rows2;
    if (a.VS > m + 1) a.VS = m + 1;
    a.rows_smem = (left - a.VS * rows2) / n2;
    if (a.rows_smem > a.rows_per_cta) a.rows_smem = a.rows_per_cta;
    // measured (random systems, restart 50, us per Arnoldi step, cluster / grid-wide kernel): n = 256 10.9 / 14.1, 512 11.2 / 14.0,
    // 600 12.0 / 16.7, 640 (four rows per CTA from L2) 13.2 / 14.2, 1024 (43 rows from L2) 26.3 / 16.7: the cluster wins
    // while (almost) all of A sits in shared memory
    if (a.rows_per_cta - a.rows_smem > CL_GB) return BIE_CLUSTER_NOT_TAKEN;
    const ClusterSmem L = cluster_smem(n, m, a.rows_per_cta, a.mp, CS, a.VS, a.rows_smem);
    a.A = A; a.lda = lda; a.n = n; a.b = rhs; a.tol = tol; a.m = m; a.max_iters = max_iters; a.x = x;
    a.iters_out = iters_out; a.relres_out = relres_out; a.status_out = status_out; a.res_hist = res_hist;
    a.Vg = Vg; a.nld = nld; a.R = R;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(CS); cfg.blockDim = dim3(CL_THREADS);
    cfg.dynamicSmemBytes = sizeof(double) * (size_t)L.total;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = CS; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    BIE_CUDA(cudaLaunchKernelEx(&cfg, bie_gmres_cluster_kernel, a));
    return BIE_OK;
}
