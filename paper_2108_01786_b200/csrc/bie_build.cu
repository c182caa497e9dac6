// bie_build.cu -- SURVEY 8(a) rows a2-a4: the dense collocation matrix of Eq. (3.16).
//
// Tiling.  A CTA of 128 threads owns a tile of T target rows x 256 source columns.  Each thread keeps the
// per-node factors of TWO adjacent source columns in registers and walks down the T target rows, whose
// factors E_t sit in shared memory and are read as warp-wide broadcasts.  A warp therefore writes,
// per target row, 32 x 16 B = 512 contiguous bytes of that row (128-bit coalesced stores, full 128 B lines).
//
// Per entry (fast path): 10 FP64-pipe instructions + 1 MUFU + 1 integer compare, no transcendental
// (bie_common.cuh, "difference form").  The walk over the target rows is split into segments of constant target
// component, so that the Re/Im selection of Eq. (3.10) and the -1/M_k of E_k become
// three per-segment register coefficients (U, W, cst):
//     entry = (U dr + W di) / den - cst,     dr + i di = E_s - E_t,   den = dr^2 + di^2,
//     U = alpha Ei_s + 2 beta Er_s,  W = 2 beta Ei_s - alpha Er_s,  cst = beta + em,
//     Im c  ->  (alpha, beta) = (-2 qi,  qr)     [k = 0, j = 0]  and  [k >= 1, j >= 1]
//     Re c  ->  (alpha, beta) = (-2 qr, -qi)     [k = 0, j >= 1]
//    -Re c  ->  (alpha, beta) = ( 2 qr,  qi)     [k >= 1, j = 0]
// The inner loop has no branch: it only tracks the smallest high word of den per column (the generic loop: ORs a "near"
// flag, den < thr_s, which includes s == t).  After every BUILD_RB rows the warp votes; if any lane saw a near pair, those
// rows are revisited and the near entries are overwritten with the Laurent-series value, or with the precomputed diagonal
// entry when s == t.  Whole blocks of rows of a warp whose columns all lie inside the matrix take the FAST row
// loop (no row clamp, no store predicate, the row pointer advanced by additions: 18.7 issued instructions per entry instead
// of 26); tails, the last warp of a ragged matrix and the block format of the hybrid operator take the generic one.
// The grid is one-dimensional and bie_build_tile() puts the tiles that hold the diagonal first (see there).
#include "bie_common.cuh"

#define BUILD_THREADS 128
#define BUILD_COLS 2
#define BUILD_TILE_W (BUILD_THREADS * BUILD_COLS)
#ifndef BUILD_RB
#define BUILD_RB 4
#endif
#ifndef BUILD_MIN_CTAS
#define BUILD_MIN_CTAS 4      // CTAs of 128 threads per SM the register allocation must allow.  Measured at config 5 in round 1 (0.411 ms
                              // at 4): 5 -> 0.414, 6 -> 0.448, 8 -> 0.487 ms; with the fast row loop 3, 4 and 5 are within 1 % of each other
#endif

// Tile of CTA L of the one-dimensional grid.  The tiles that hold the diagonal go FIRST (two per block of T rows: the
// tile columns that the rows [t0, t0 + T) can meet, T <= 256): their near entries take the slow path, which makes
// such a CTA several times slower than the others -- in launch order the ones of the last wave finished 50 us after
// everything else at n = 16384 (0.41 ms with them anywhere, 0.35 ms without the near path; measured).  The other tiles
// keep the row-major order (x fastest), so that concurrently running CTAs write the same rows.
__device__ __forceinline__ void bie_build_tile(int L, int gx, int gy, int T, int& bx, int& by)
{
    if (gx < 3) { bx = L % gx; by = L / gx; return; }
    int j;
    if (L < 2 * gy) { by = L >> 1; j = L & 1; }
    else { const int r = L - 2 * gy; by = r / (gx - 2); j = 2 + r % (gx - 2); }
    bx = (int)(((long long)by * T / BUILD_TILE_W + j) % gx);
}

struct SrcCol {
    double er, ei;      // E_s
    int thi;            // high word of thr_s
    double u, w, cst;   // per-segment coefficients
};

__device__ __forceinline__ double bie_entry_fast(const SrcCol& s, const double2 te, int& flag)
{
    const double dr = s.er - te.x, di = s.ei - te.y;
    const double den = fma(dr, dr, di * di);
    const double val = fma(s.w, di, s.u * dr);
    flag |= (__double2hiint(den) < s.thi) ? 1 : 0;
    return fma(val, bie_rcp3(den), -s.cst);
}

// the same entry; instead of a flag the smallest high word of den seen so far (one integer min per entry; the near
// test den < thr_s is made once per block of rows)
__device__ __forceinline__ double bie_entry_fast_min(const SrcCol& s, const double2 te, int& mn)
{
    const double dr = s.er - te.x, di = s.ei - te.y;
    const double den = fma(dr, dr, di * di);
    const double val = fma(s.w, di, s.u * dr);
    mn = min(mn, __double2hiint(den));
    return fma(val, bie_rcp3(den), -s.cst);
}

// exact value of a near entry (rare): Laurent series from the coordinate differences, or the diagonal limit
static __device__ __noinline__ double bie_entry_near(const double2* __restrict__ DG, const double2* __restrict__ XY,
                                                     double sa, double sb, double sem, int sidx, int tidx)
{
    if (sidx == tidx) return DG[tidx].x;
    const double2 zs = XY[sidx], zt = XY[tidx];
    double cr, ci;
    bie_cot_half_near(zs.x - zt.x, zs.y - zt.y, &cr, &ci);
    // entry = alpha X/den + beta Y/den with cot = (-2X + iY)/den
    return fma(sb, ci, -0.5 * sa * cr) - sem;
}

// (alpha, beta) of the block (source on Gamma_0?, target on Gamma_0?) for the source weight q (bie_common.cuh)
__device__ __forceinline__ void bie_block_coef(bool src0, bool tgt0, double qr, double qi, double& al, double& be)
{
    if (src0 == tgt0) { al = -2.0 * qi; be = qr; }       // Im c
    else if (tgt0)    { al = -2.0 * qr; be = -qi; }      // Re c   (G_0j)
    else              { al = 2.0 * qr;  be = qi; }       // -Re c  (-G_k0)
}

// rows [ta, tb) of a thread that saw a near pair: its near entries are overwritten with the exact value
static __device__ __forceinline__ void bie_build_fix_near(const NodeTable& nt, const SrcCol* src, const int* scomp, const double* sqr,
                                                       const double* sqi, const double* sem, const double2* sE, int t0, int ta, int tb,
                                                       int k, int s0, int ncols, double* A, long long lda, int nchT, bool tiled)
{
    for (int t = ta; t < tb; ++t) {
        const double2 te = sE[t - t0];
#pragma unroll
        for (int c = 0; c < BUILD_COLS; ++c) {
            if (s0 + c >= ncols) continue;
            const double dr = src[c].er - te.x, di = src[c].ei - te.y;
            const double den = fma(dr, dr, di * di);
            if (__double2hiint(den) < src[c].thi) {
                double al, be;
                bie_block_coef(scomp[c] == 0, k == 0, sqr[c], sqi[c], al, be);
                A[bie_entry_off(tiled ? 0 : lda, nchT, t, s0 + c)] =
                    bie_entry_near(nt.DG, nt.XY, al, be, (scomp[c] == k) ? sem[c] : 0.0, s0 + c, t);
            }
        }
    }
}

// TILED: A is the block format of the hybrid operator (bie_common.cuh) instead of row-major with leading dimension lda
template <bool TILED>
__global__ void __launch_bounds__(BUILD_THREADS, BUILD_MIN_CTAS)
bie_build_kernel(NodeTable nt, CompTable ct, double* __restrict__ A, long long lda, int T, int only0, int ncols, int nrows, int gx, int gy)
{
    extern __shared__ __align__(16) double2 sm[];  // [T] E_t
    int bx, by;
    bie_build_tile(blockIdx.x, gx, gy, T, bx, by);
    const int c0 = bx * BUILD_TILE_W;
    const int t0 = by * T;
    const int t1 = min(t0 + T, nrows);      // nrows = n, or the rows of the hybrid operator's block
    if (only0 && t0 >= ct.off[1] && c0 >= ct.off[1]) return;  // a4: solid-solid tiles stay
    double2* sE = sm;
    for (int i = threadIdx.x; i < t1 - t0; i += BUILD_THREADS) sE[i] = nt.E[t0 + i];
    const int s0 = c0 + BUILD_COLS * threadIdx.x;  // < npad by construction
    SrcCol src[BUILD_COLS];
    double sqr[BUILD_COLS], sqi[BUILD_COLS], sem[BUILD_COLS];
    int scomp[BUILD_COLS];
#pragma unroll
    for (int c = 0; c < BUILD_COLS; ++c) {
        const double2 e = nt.E[s0 + c], mt = nt.MT[s0 + c], q = nt.Q[s0 + c];
        src[c].er = e.x; src[c].ei = e.y;
        src[c].thi = __double2hiint(mt.y);
        sqr[c] = q.x; sqi[c] = q.y;
        sem[c] = nt.DG[s0 + c].y;
        scomp[c] = nt.COMP[s0 + c];
    }
    __syncthreads();
    const bool full = (s0 + 1 < ncols);   // ncols = n, or the width of the hybrid operator's block
    const bool part = (s0 < ncols);
    const bool wfull = __all_sync(0xffffffffu, full);   // warp-uniform: the fast row loop votes per block of rows
    const int nchT = (ncols + BIE_TILE_COLS - 1) / BIE_TILE_COLS;   // block format (lda == 0)
    for (int k = 0; k < ct.ncomp; ++k) {
        const int a = max(t0, ct.off[k]), b = min(t1, ct.off[k + 1]);
        if (a >= b) continue;
#pragma unroll
        for (int c = 0; c < BUILD_COLS; ++c) {
            double al, be;
            bie_block_coef(scomp[c] == 0, k == 0, sqr[c], sqi[c], al, be);
            src[c].u = fma(al, src[c].ei, 2.0 * be * src[c].er);
            src[c].w = fma(-al, src[c].er, 2.0 * be * src[c].ei);
            src[c].cst = be + ((scomp[c] == k) ? sem[c] : 0.0);
        }
        int tb = a;
        if (!TILED && wfull) {
            // whole blocks of BUILD_RB rows, both columns of every lane inside the matrix (all but the last warp of the last tile
            // column): no clamp, no store predicate, the row pointer advanced by additions -- 17 instead of 26 issued
            // instructions per entry (the kernel is issue-bound before it is write-bound)
            double* p = A + (long long)a * lda + s0;
            const double2* se = sE + (a - t0);
            for (; tb + BUILD_RB <= b; tb += BUILD_RB, p += BUILD_RB * lda, se += BUILD_RB) {
                int m0 = 0x7fffffff, m1 = 0x7fffffff;
#pragma unroll
                for (int r = 0; r < BUILD_RB; ++r) {
                    const double2 te = se[r];
                    const double e0 = bie_entry_fast_min(src[0], te, m0);
                    const double e1 = bie_entry_fast_min(src[1], te, m1);
                    *reinterpret_cast<double2*>(p + (long long)r * lda) = make_double2(e0, e1);
                }
                const int flag = (m0 < src[0].thi) | (m1 < src[1].thi);
                if (__any_sync(0xffffffffu, flag)) {
                    if (flag) bie_build_fix_near(nt, src, scomp, sqr, sqi, sem, sE, t0, tb, tb + BUILD_RB, k, s0, ncols, A, lda, nchT, false);
                }
            }
        }
        for (; tb < b; tb += BUILD_RB) {
            int flag = 0;
            double* row = TILED ? A : A + (long long)tb * lda + s0;
#pragma unroll
            for (int r = 0; r < BUILD_RB; ++r) {
                const int t = min(tb + r, b - 1);  // the tail repeats the last row (same values, same address)
                const double2 te = sE[t - t0];
                const double e0 = bie_entry_fast(src[0], te, flag);
                const double e1 = bie_entry_fast(src[1], te, flag);
                double* p = TILED ? A + bie_entry_off(0, nchT, t, s0) : row + (long long)(t - tb) * lda;
                if (full) *reinterpret_cast<double2*>(p) = make_double2(e0, e1);
                else if (part) p[0] = e0;
            }
            if (__any_sync(0xffffffffu, flag)) {
                if (flag) bie_build_fix_near(nt, src, scomp, sqr, sqi, sem, sE, t0, tb, min(tb + BUILD_RB, b), k, s0, ncols, A, lda, nchT, TILED);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// Vortex-sheet variant (BIE_VARIANT_VORTEX) and normal-velocity operator: the matrix S of Eqs. (4.14) + (4.17) from
// the adjoint matrices of Eq. (4.7), (K+_jk)_ml = K_jk(alpha_jl, alpha_km)/M_j.  Entry of row
// t = (k,m), column s = (j,l):   c+ = zeta'_t/(2 M_j) cot((zeta_t - zeta_s)/2) = -(u_t/M_j)(-2X + iY)/den,
// u_t = zeta'_t/2, i.e. the weight comes from the ROW node and only 1/M_j from the column.  With m_s = 1/M_j folded
// into the source's factors (X' = m_s X, Y' = m_s (M_s - M_t)) the entry is (A_t X' + B_t Y')/den with
//     Im c+ -> (A, B) = (2 u_i, -u_r)   [k = 0, j = 0: 1/2 I + K+_00]  and  [k, j >= 1: -1/2 I + K+_jk]
//    -Re c+ -> (-2 u_r, -u_i)           [k = 0, j >= 1: -G+_j0]
//     Re c+ -> ( 2 u_r,  u_i)           [k >= 1, j = 0:  G+_0k]
// 11 FP64-pipe instructions per entry in the row-side difference form (bie_entry_fast_dagger); the row constants (U, W, B) sit
// in shared memory per target row, one set for columns on Gamma_0 and one for columns on solids.  Same tiling, near-pair
// handling and stores as bie_build_kernel.
struct SrcColD {
    double er, ei;        // E_s
    double ms;            // 1 / M_j
    int thi;
};

// (A_t, B_t) of the row's weight u_t = zeta'_t / 2 for a column on Gamma_0 (col0) or on a solid:
//   normal-velocity operator (kap): -G+_00 (3.24) ; K+_j0 (3.19)      row on Gamma_0: K+_00 ; -G+_j0      row on a solid: G+_0k ; K+_jk
__device__ __forceinline__ double2 bie_dagger_ab(bool kap, bool row0, bool col0, double ur, double ui)
{
    const double2 im = make_double2(2.0 * ui, -ur);
    if (kap)  return col0 ? make_double2(-2.0 * ur, -ui) : im;
    if (row0) return col0 ? im : make_double2(-2.0 * ur, -ui);
    return col0 ? make_double2(2.0 * ur, ui) : im;
}

// Row-side difference form (bie_common.cuh): with d = E_s - E_t,  X = Ei_t dr - Er_t di,  Y = 2 (Er_t dr + Ei_t di) + den, so
//     (A_t X + B_t Y)/den = (U_t dr + W_t di)/den + B_t,     U_t = A_t Ei_t + 2 B_t Er_t,   W_t = 2 B_t Ei_t - A_t Er_t,
// row constants per column class; 11 FP64-pipe instructions per entry (13 with the (X, Y) form).
__device__ __forceinline__ double bie_entry_fast_dagger(const SrcColD& s, const double2 te, const double2 uw, const double bt, int& flag)
{
    const double dr = s.er - te.x, di = s.ei - te.y;
    const double den = fma(dr, dr, di * di);
    const double num = fma(uw.y, di, uw.x * dr);
    flag |= (__double2hiint(den) < s.thi) ? 1 : 0;
    return fma(num, bie_rcp3(den), bt) * s.ms;
}

// rows [ta, tb) of a thread that saw a near pair: its near entries are overwritten with the exact value
static __device__ __forceinline__ void bie_dagger_fix_near(const NodeTable& nt, const CompTable& ct, const SrcColD* src, const bool* col0,
                                                           const bool* kap, const double2* sE, const double* sK, int dmin, int t0, int ta,
                                                           int tb, int s0, int ncols, double* A, long long lda, int nchT, bool tiled, bool nv)
{
    for (int t = ta; t < tb; ++t) {
        const double2 te = sE[t - t0];
#pragma unroll
        for (int c = 0; c < BUILD_COLS; ++c) {
            if (s0 + c >= ncols) continue;
            const double dr = src[c].er - te.x, di = src[c].ei - te.y;
            const double den = fma(dr, dr, di * di);
            if (__double2hiint(den) < src[c].thi) {
                const int k = nt.COMP[t];
                const double Mk = (double)(ct.off[k + 1] - ct.off[k]);
                const double2 q = nt.Q[t];
                const double2 ab = bie_dagger_ab(nv, k == 0, col0[c], q.x * Mk, q.y * Mk);
                // (A X' + B Y')/den with cot = (-2X + iY)/den; the diagonal entry is prepared per node
                double v = bie_entry_near(nt.DG, nt.XY, src[c].ms * ab.x, src[c].ms * ab.y, 0.0, s0 + c, t);
                if (kap[c]) v += sK[t - s0 - c - dmin];
                A[bie_entry_off(tiled ? 0 : lda, nchT, t, s0 + c)] = v;
            }
        }
    }
}

// the same entry with the smallest high word of den instead of a flag (bie_entry_fast_min)
__device__ __forceinline__ double bie_entry_fast_dagger_min(const SrcColD& s, const double2 te, const double2 uw, const double bt, int& mn)
{
    const double dr = s.er - te.x, di = s.ei - te.y;
    const double den = fma(dr, dr, di * di);
    const double num = fma(uw.y, di, uw.x * dr);
    mn = min(mn, __double2hiint(den));
    return fma(num, bie_rcp3(den), bt) * s.ms;
}

// shared memory of bie_build_dagger_kernel in bytes (kap: with the two copies of the real-cot table)
static inline size_t bie_dagger_smem(int T, bool kap)
{
    return 4 * sizeof(double2) * (size_t)T + (kap ? sizeof(double) * (2 * (size_t)(T + BUILD_TILE_W) + 2) : 0) + 16;
}

template <bool TILED>
__global__ void __launch_bounds__(BUILD_THREADS)
bie_build_dagger_kernel(NodeTable nt, CompTable ct, double* __restrict__ A, long long lda, int T, int only0, int ncols, int nrows,
                        const double* __restrict__ kappa /* NULL: vortex-sheet S; else the normal-velocity operator */, int gx, int gy)
{
    // [T] E_t, [T] (U,W) for columns on Gamma_0, [T] (U,W) for solids, [T] B for Gamma_0 columns, [T] B for solids,
    // [T + 256] kappa (KA), [T + 258] kappa shifted by one (KB[x] = KA[x - 1])
    extern __shared__ __align__(16) double2 sm[];
    int bx, by;
    bie_build_tile(blockIdx.x, gx, gy, T, bx, by);
    const int c0 = bx * BUILD_TILE_W;
    const int t0 = by * T;
    const int t1 = min(t0 + T, nrows);   // n; M_0 for the normal-velocity operator (rows on Gamma_0 only); the block's rows
    if (only0 && t0 >= ct.off[1] && c0 >= ct.off[1]) return;
    double2* sE = sm;
    double2* sUW0 = sm + T;
    double2* sUW1 = sm + 2 * T;
    double* sB0 = reinterpret_cast<double*>(sm + 3 * T);
    double* sB1 = sB0 + T;
    double* sK = reinterpret_cast<double*>(sm + 4 * T);          // KA
    double* sKB = sK + (T + BUILD_TILE_W);
    const int M0 = ct.off[1];
    for (int i = threadIdx.x; i < t1 - t0; i += BUILD_THREADS) {
        const int t = t0 + i;
        const int k = nt.COMP[t];
        const double Mk = (double)(ct.off[k + 1] - ct.off[k]);
        const double2 q = nt.Q[t], e = nt.E[t];
        const double ur = q.x * Mk, ui = q.y * Mk;   // zeta'_t / 2
        const double2 ab0 = bie_dagger_ab(kappa != nullptr, k == 0, true, ur, ui);
        const double2 ab1 = bie_dagger_ab(kappa != nullptr, k == 0, false, ur, ui);
        sE[i] = e;
        sUW0[i] = make_double2(fma(ab0.x, e.y, 2.0 * ab0.y * e.x), fma(-ab0.x, e.x, 2.0 * ab0.y * e.y));
        sUW1[i] = make_double2(fma(ab1.x, e.y, 2.0 * ab1.y * e.x), fma(-ab1.x, e.x, 2.0 * ab1.y * e.y));
        sB0[i] = ab0.y; sB1[i] = ab1.y;
    }
    // the real-cot table of the Gamma_0 - Gamma_0 block of the normal-velocity operator: kappa_{(t - s) mod M_0} for the tile's
    // differences d = t - s in [t0 - c0 - 255, t1 - 1 - c0].  Entry (t, s0) takes KA[i], entry (t, s0 + 1) takes KA[i - 1],
    // i = t - s0 - dmin >= 1: for odd i the pair is an aligned double2 of KA, for even i of the shifted copy KB -- one
    // 128-bit load per row and thread, consecutive lanes on consecutive 16 bytes (two 64-bit loads at a 16-byte stride
    // have two-way bank conflicts)
    const int dmin = t0 - c0 - (BUILD_TILE_W - 1);
    const bool have_k = (kappa != nullptr && c0 < M0);
    if (have_k)
        for (int i = threadIdx.x; i < (t1 - t0) + BUILD_TILE_W - 1; i += BUILD_THREADS) {
            int d = (dmin + i) % M0;
            if (d < 0) d += M0;
            const double kv = __ldg(kappa + d);
            sK[i] = kv; sKB[i + 1] = kv;
        }
    const int s0 = c0 + BUILD_COLS * threadIdx.x;  // < npad by construction
    SrcColD src[BUILD_COLS];
    bool col0[BUILD_COLS], kap[BUILD_COLS];
#pragma unroll
    for (int c = 0; c < BUILD_COLS; ++c) {
        const double2 e = nt.E[s0 + c], mt = nt.MT[s0 + c];
        const int j = nt.COMP[s0 + c];
        src[c].ms = (j >= 0) ? 1.0 / (double)(ct.off[j + 1] - ct.off[j]) : 0.0;
        src[c].er = e.x; src[c].ei = e.y;
        src[c].thi = __double2hiint(mt.y);
        col0[c] = (j == 0);
        kap[c] = (kappa != nullptr && j == 0);
    }
    const bool same_cls = (col0[0] == col0[1]);
    __syncthreads();
    const bool full = (s0 + 1 < ncols);
    const bool part = (s0 < ncols);
    const int nchT = (ncols + BIE_TILE_COLS - 1) / BIE_TILE_COLS;   // block format (lda == 0)
    const double2* sUWa = col0[0] ? sUW0 : sUW1;
    const double2* sUWb = col0[1] ? sUW0 : sUW1;
    const double* sBa = col0[0] ? sB0 : sB1;
    const double* sBb = col0[1] ? sB0 : sB1;
    int tb = t0;
    if (!TILED && __all_sync(0xffffffffu, full && same_cls)) {
        // whole blocks of BUILD_RB rows; both columns of every lane inside the matrix and on the same side of M_0 (all warps
        // but the one that holds column M_0 - 1 when M_0 is odd, and the last one of a ragged matrix): one set of row constants
        // per row, no clamp, no store predicate, the row pointer advanced by additions
        double* p = A + (long long)t0 * lda + s0;
        const bool kp = kap[0];
        const int i0 = t0 - s0 - dmin;
        const double2* kx = reinterpret_cast<const double2*>((i0 & 1) ? sK : sKB);    // rows with even r
        const double2* ky = reinterpret_cast<const double2*>((i0 & 1) ? sKB : sK);    // rows with odd r
        for (; tb + BUILD_RB <= t1; tb += BUILD_RB, p += BUILD_RB * lda) {
            int m0 = 0x7fffffff, m1 = 0x7fffffff;
#pragma unroll
            for (int r = 0; r < BUILD_RB; ++r) {
                const int i = tb - t0 + r;
                const double2 te = sE[i];
                const double2 uw = sUWa[i];
                const double bt = sBa[i];
                double e0 = bie_entry_fast_dagger_min(src[0], te, uw, bt, m0);
                double e1 = bie_entry_fast_dagger_min(src[1], te, uw, bt, m1);
                if (kp) {
                    const double2 kv = ((r & 1) ? ky : kx)[(i0 + i) >> 1];
                    e0 += kv.y; e1 += kv.x;
                }
                *reinterpret_cast<double2*>(p + (long long)r * lda) = make_double2(e0, e1);
            }
            const int flag = (m0 < src[0].thi) | (m1 < src[1].thi);
            if (__any_sync(0xffffffffu, flag)) {
                if (flag) bie_dagger_fix_near(nt, ct, src, col0, kap, sE, sK, dmin, t0, tb, tb + BUILD_RB, s0, ncols, A, lda, nchT, false, kappa != nullptr);
            }
        }
    }
    for (; tb < t1; tb += BUILD_RB) {
        int flag = 0;
        double* row = TILED ? A : A + (long long)tb * lda + s0;
#pragma unroll
        for (int r = 0; r < BUILD_RB; ++r) {
            const int t = min(tb + r, t1 - 1);  // the tail repeats the last row (same values, same address)
            const double2 te = sE[t - t0];
            const double2 uwa = sUWa[t - t0];
            const double2 uwb = same_cls ? uwa : sUWb[t - t0];   // both columns on the same side of M_0, almost always
            double e0 = bie_entry_fast_dagger(src[0], te, uwa, sBa[t - t0], flag);
            double e1 = bie_entry_fast_dagger(src[1], te, uwb, sBb[t - t0], flag);
            if (kap[0]) e0 += sK[t - s0 - dmin];
            if (kap[1]) e1 += sK[t - s0 - 1 - dmin];
            double* p = TILED ? A + bie_entry_off(0, nchT, t, s0) : row + (long long)(t - tb) * lda;
            if (full) *reinterpret_cast<double2*>(p) = make_double2(e0, e1);
            else if (part) p[0] = e0;
        }
        if (__any_sync(0xffffffffu, flag)) {
            if (flag) bie_dagger_fix_near(nt, ct, src, col0, kap, sE, sK, dmin, t0, tb, min(tb + BUILD_RB, t1), s0, ncols, A, lda, nchT, TILED, kappa != nullptr);
        }
    }
}

// the first ncols columns of the first nrows rows are written (nrows = ncols = n: the whole matrix; nrows <= 0: all rows)
int bie_launch_build(bie_ctx* ctx, double* A, int64_t lda, int ncols, int nrows, int only_comp0, cudaStream_t st)
{
    if (!ctx || !A) return BIE_ERR_NULL;
    if (!ctx->have_geom) return BIE_ERR_GEOMETRY;
    const int n = ctx->n;
    if (ncols < 1 || ncols > n || nrows > n) return BIE_ERR_ARG;
    // lda == 0: the block format of the hybrid operator (bie_common.cuh), square blocks only
    if (lda == 0 ? (nrows != ncols) : (lda < ncols || (lda & 1))) return BIE_ERR_LAYOUT;
    if (((uintptr_t)A) & 15u) return BIE_ERR_LAYOUT;
    const NodeTable nt = bie_node_table(ctx);
    const int gx = (ncols + BUILD_TILE_W - 1) / BUILD_TILE_W;
    int nt_rows = nrows > 0 ? nrows : n;
    if (ctx->variant == BIE_VARIANT_NORMAL_INTERNAL) nt_rows = ctx->counts[0];   // M_0 x n: rows on Gamma_0 only
    const bool dagger = (ctx->variant == BIE_VARIANT_VORTEX || ctx->variant == BIE_VARIANT_NORMAL_INTERNAL);
    // rows per CTA: 128 when that still gives every SM several CTAs, else smaller ...
    int T = 128;
    while (T > 8 && (long long)gx * ((nt_rows + T - 1) / T) < 4LL * ctx->sm_count) T >>= 1;
    // ... and, for grids of several waves, the T in [96, 256] that fills whole waves of resident CTAs: the tail wave
    // of the default (8192 CTAs = 11.07 waves of 740 at n = 16384) cost 16 % (profiles/r01b_ncu_full_cfg5.md)
    {
        int occ = 0;
        if (dagger) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, bie_build_dagger_kernel<false>, BUILD_THREADS, bie_dagger_smem(256, ctx->variant == BIE_VARIANT_NORMAL_INTERNAL));
        else cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, bie_build_kernel<false>, BUILD_THREADS, 2 * 8 * 256 + 16);
        const long long wave = (long long)ctx->sm_count * (occ > 0 ? occ : 1);
        if ((long long)gx * ((nt_rows + 127) / 128) >= 2 * wave) {
            double best = 0.0;
            for (int t = 96; t <= 256; t += BUILD_RB) {
                const long long gy = (nt_rows + t - 1) / t, ctas = (long long)gx * gy;
                const double eff = (double)ctas / (double)(((ctas + wave - 1) / wave) * wave) * (double)nt_rows / (double)(gy * t);
                if (eff > best + 1e-9) { best = eff; T = t; }
            }
        }
    }
    const int gy = (nt_rows + T - 1) / T;
    const unsigned grid = (unsigned)gx * (unsigned)gy;     // one-dimensional: bie_build_tile orders the tiles
    const bool tiled = (lda == 0);
    const double* kap = ctx->variant == BIE_VARIANT_NORMAL_INTERNAL ? ctx->kappa : nullptr;
    if (dagger) {
        const size_t sm = bie_dagger_smem(T, kap != nullptr);
        if (tiled) bie_build_dagger_kernel<true><<<grid, BUILD_THREADS, sm, st>>>(nt, ctx->comps, A, 0, T, only_comp0, ncols, nt_rows, kap, gx, gy);
        else bie_build_dagger_kernel<false><<<grid, BUILD_THREADS, sm, st>>>(nt, ctx->comps, A, (long long)lda, T, only_comp0, ncols, nt_rows, kap, gx, gy);
    } else {
        const size_t sm = sizeof(double2) * T + 16;
        if (tiled) bie_build_kernel<true><<<grid, BUILD_THREADS, sm, st>>>(nt, ctx->comps, A, 0, T, only_comp0, ncols, nt_rows, gx, gy);
        else bie_build_kernel<false><<<grid, BUILD_THREADS, sm, st>>>(nt, ctx->comps, A, (long long)lda, T, only_comp0, ncols, nt_rows, gx, gy);
    }
    BIE_CUDA(cudaGetLastError());
    return BIE_OK;
}
