// bie_free.cuh -- matrix-free form of SURVEY 8(a) row a6: y_t = sum_s A[t][s] x_s with the entries of
// Eq. (3.16) recomputed on the fly from the node tables; no matrix traffic at all.
// Device functions shared by bie_matvec_free (bie_matvec.cu) and the matrix-free / hybrid GMRES (bie_gmres.cu).
//
// Arithmetic ("difference form", bie_common.cuh).  With E = e^{i zeta} per node, d = E_s - E_t = dr + i di,
// den = |d|^2 and the block coefficients (alpha, beta) of Eq. (3.10), the product of an entry with x_s is
//     A[t][s] x_s = (alpha X + beta Y) x_s / den = ( U_s dr + W_s di ) / den - beta_s x_s,
//     U_s = x_s (alpha Ei_s + 2 beta Er_s),   W_s = x_s (2 beta Ei_s - alpha Er_s),
// so everything that depends on the source alone is folded, once per matvec and per source (O(n)), into ONE
// double2 (U, W) per target class (class 0: target on Gamma_0, class 1: target on a solid; the class fixes
// the Re/Im/sign selection of Eq. (3.10)), and the constant -sum_s beta_s x_s (one number per
// class and application) is subtracted by the row owner.  Per pair that leaves 10 FP64-pipe instructions:
// 2 sub, 2 for den, 2 for the numerator, 3 FMA refining MUFU.RCP64H (bie_rcp3), 1 FMA accumulating.
//
// Work split.  The rows are cut into row blocks of FREE_ROWS = 128 targets of one class; the (row block x source)
// rectangle list is laid out linearly and cut into gridDim.x equal slabs, one per CTA, so every SM has the same
// number of pairs whatever n is.  A CTA's slab touches one or two row blocks ("parts"); for each part the
// warps share the part's sources, every lane keeps FREE_NT = 4 targets of the block in registers and runs over
// its warp's sources, which the warp stages 32 at a time in its own shared-memory buffer (no CTA-wide barrier in
// the pair loop) and reads as warp-wide broadcasts.  The warp sums are added in fixed order and go to a
// partial buffer in global memory (L2); after a grid barrier the owner of a row adds the (at most three)
// partials of its row block, again in fixed order: the result is deterministic.
//
// Hybrid operator (s_off > 0).  The leading s_off x s_off block of the matrix is STORED and streamed by the caller
// (bie_gmres.cu, bie_gemv.cuh "block ring"); this operator supplies the rest, an L-shaped region: row blocks below
// s_off (s_off is a row-block boundary) take the sources [s_off, n), the others all sources.
//
// Near pairs.  den < taubar M_t (den/M_t = |e^{iw} - 1|^2 ~ |w|^2; this includes s == t) marks a pair as near:
// it is left out of the fast sum by predication, and its exact entry (Laurent series of cot, or the analytic
// diagonal limit PAPER.md:L265) comes from the sparse near matrix that bie_near.cu builds once per geometry;
// the owner of a row adds  sum_k val[k] x[col[k]]  when it gathers the partials (val = entry + beta_s: the
// constant term above runs over ALL sources).  The rank-one E_k is applied there too, as
// -(1/M_k) sum_{s in k} x_s.
#pragma once
#include "bie_common.cuh"

#define FREE_THREADS 512
#ifndef FREE_SRC_UNROLL_N
#define FREE_SRC_UNROLL_N 2
#endif
constexpr int FREE_SRC_UNROLL = FREE_SRC_UNROLL_N;   // sources per unrolled step of the pair loop
#define FREE_WARPS (FREE_THREADS / 32)
#define FREE_NT 4
#define FREE_ROWS (32 * FREE_NT)

// host-computed description of the work split (by value into the kernels)
struct FreePlan {
    int M0;          // rows of class 0 = nodes of component 0
    int NB0, NB;     // row blocks of class 0, all row blocks
    int nb_below;    // row blocks entirely below s_off (hybrid operator; 0 otherwise)
    int UBb, UBf;    // one-directional list: units (of 2 sources) of a block below s_off, (npad - s_off) / 2, and of the others, npad / 2
    long long U;     // list length: nb_below UBb + (NB - nb_below) UBf, or the sources of the symmetric list
    int Geff;        // CTAs that take a slab (<= gridDim.x)
    int sym;         // 1: symmetric (oddness) work split of bie_free_sym.cuh: U = sources of the triangular list, PC valid
    double* PC;      // sym: [NB][npad] reverse partial sums (row block I, source s)
    const long long* sym_cum;   // sym: [NB + 1] sources before position k of the (permuted) triangular list
    const int* sym_perm;        // sym: [NB] row block at position k
    const int* sym_pos;         // sym: [NB] position of row block b
    int vortex;      // 1: the vortex-sheet matrix S (BIE_VARIANT_VORTEX) instead of Eq. (3.16); see free_parts
    int s_off;       // hybrid operator: the leading s_off x s_off block comes from the caller's stored block (0: none)
    int stage_buf;   // doubles of one staging buffer of a warp (free_stage_buf_doubles): fixes the shared-memory strides
    double2* T;      // [2][npad]: (U,W) class 0, (U,W) class 1     (vortex: (P,Q) = mu E, (R,B) = mu (M, 1))
    double* SB;      // [2][4][FREE_SB_LD] per-CTA partials of sum_s beta_s x_s: class 0 / 1 over s >= s_off, class 0 / 1 over s < s_off;
                     // two copies (sb_sel): an application may write its constants while other CTAs still gather the previous one's
    double* PB;      // [(NB + Geff)][FREE_ROWS] partial sums, part id = list position of the row block + CTA
    const double* taubar;     // device scalar: near threshold relative to M_t (bie_near.cu)
    const int* near_ptr;      // CSR near matrix: offsets of the (row, segment) lists, row t = [ptr[8t], ptr[8t+8])
    const int* near_col;
    const double* near_val;
};
#define FREE_SB_LD 256   // >= gridDim.x (one CTA per SM, <= 256 SMs)

// doubles of shared scratch, in this order: warp sums [16][128]; component sums [2][BIE_MAX_COMP] and the four constants;
// warp staging buffers [16][2 stages] of 32 sources: E, (U,W) (and (R,B) for the vortex-sheet matrix) as double2, and
// the near thresholds of the symmetric loops as int; reverse-sum slots of bie_free_sym.cuh
#define FREE_CSUM_DOUBLES (2 * BIE_MAX_COMP + 4)
#define FREE_HEAD_DOUBLES (FREE_WARPS * FREE_ROWS + FREE_CSUM_DOUBLES)
#ifndef SYM_BATCH
#define SYM_BATCH 8
#endif
#ifndef SYM_PART_PAD
#define SYM_PART_PAD 144      // symmetric work list: every row block's list is longer by this many VIRTUAL sources (no work): the fixed
                              // cost of starting a list (target loads, exposed first loads of its segments, warp-sum reduction) is
                              // 2.3-2.7 us = the time of 125-145 sources (least-squares fit of the CTAs' pair-loop times to their
                              // sources and list starts, config 5), so that cutting the list into equal slabs equalises TIME
#endif
#define SYM_COL_STRIDE 33                                         // [SYM_BATCH][33] doubles per warp: lane-private slots, no bank conflicts
#define SYM_COL_DOUBLES (FREE_WARPS * SYM_BATCH * SYM_COL_STRIDE)
// one staging buffer of a warp (32 sources): E and (U,W) as double2; + (R,B) for the vortex-sheet matrix
__host__ __device__ inline int free_stage_buf_doubles(bool vortex, bool /*sym*/) { return vortex ? 192 : 128; }
// shared scratch of the operator: head, [16 warps][2 buffers] staging, and the reverse-sum slots of the symmetric loops
__host__ __device__ inline int free_scratch_doubles(bool vortex, bool sym)
{
    return FREE_HEAD_DOUBLES + FREE_WARPS * 2 * free_stage_buf_doubles(vortex, sym) + (sym ? SYM_COL_DOUBLES : 0);
}

__device__ __forceinline__ long long free_slab_start(const FreePlan& fp, int c)
{
    return (long long)c * fp.U / fp.Geff;
}
__device__ __forceinline__ int free_block_row0(const FreePlan& fp, int b)
{
    return b < fp.NB0 ? b * FREE_ROWS : fp.M0 + (b - fp.NB0) * FREE_ROWS;
}
__device__ __forceinline__ int free_block_rows(const FreePlan& fp, int b, int n)
{
    const int r0 = free_block_row0(fp, b);
    const int end = b < fp.NB0 ? fp.M0 : n;
    return min(FREE_ROWS, end - r0);
}
// one-directional list: first unit of row block b, and the block that holds unit u
__device__ __forceinline__ long long free_list_start(const FreePlan& fp, int b)
{
    return b <= fp.nb_below ? (long long)b * fp.UBb : (long long)fp.nb_below * fp.UBb + (long long)(b - fp.nb_below) * fp.UBf;
}
__device__ __forceinline__ int free_list_block(const FreePlan& fp, long long u)
{
    const long long ub = (long long)fp.nb_below * fp.UBb;
    return u < ub ? (int)(u / fp.UBb) : fp.nb_below + (int)((u - ub) / fp.UBf);
}

// ---- step 1: per-source tables for the vector v (rows [r0, r1) of this CTA; v indexed from r0) ------------
// Also leaves this CTA's shares of sum_s beta_s x_s (per class; s >= s_off and s < s_off) in fp.SB.
// red: shared, >= 128 doubles.  All threads of the CTA must call; no barrier at the end (the caller's next barrier orders `red`).
__device__ __forceinline__ void free_write_tables(const NodeTable& nt, const CompTable& ct, const FreePlan& fp, int r0,
                                                  int r1, const double* v /* shared or global, v[s - r0] */, double* red, int sb_sel = 0)
{
    const int np = nt.npad;
    double sb[4] = {0.0, 0.0, 0.0, 0.0};
    for (int s = r0 + threadIdx.x; s < r1; s += blockDim.x) {
        const double2 e = nt.E[s], q = nt.Q[s];
        const double x = v[s - r0];
        if (fp.vortex) {   // S: the source only carries mu_s = x_s / M_j (the weight zeta' belongs to the ROW, Eq. 4.7)
            const double M = nt.MT[s].x;
            const int j = nt.COMP[s];
            const double mu = x / (double)(ct.off[j + 1] - ct.off[j]);
            fp.T[s]      = make_double2(mu * e.x, mu * e.y);
            fp.T[np + s] = make_double2(mu * M, mu);
            continue;
        }
        const bool src0 = (nt.COMP[s] == 0);
        // (alpha, beta): Im c -> (-2 qi, qr), Re c -> (-2 qr, -qi), -Re c -> (2 qr, qi)   (bie_common.cuh)
        double a0, b0, a1, b1;
        if (src0) { a0 = -2.0 * q.y; b0 = q.x;  a1 = 2.0 * q.x;  b1 = q.y; }   // K_00 ; -G_k0
        else      { a0 = -2.0 * q.x; b0 = -q.y; a1 = -2.0 * q.y; b1 = q.x; }   // G_0j ; K_kj
        a0 *= x; b0 *= x; a1 *= x; b1 *= x;
        fp.T[s]      = make_double2(fma(a0, e.y, 2.0 * b0 * e.x), fma(-a0, e.x, 2.0 * b0 * e.y));
        fp.T[np + s] = make_double2(fma(a1, e.y, 2.0 * b1 * e.x), fma(-a1, e.x, 2.0 * b1 * e.y));
        if (s >= fp.s_off) { sb[0] += b0; sb[1] += b1; } else { sb[2] += b0; sb[3] += b1; }
    }
    if (fp.vortex) return;
    // fixed-order sum over the CTA: lanes by shuffle, warps by threads 0..3
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
#pragma unroll
    for (int q = 0; q < 4; ++q) sb[q] = bie_warp_sum(sb[q]);
    __syncthreads();
    if (lane == 0) {
#pragma unroll
        for (int q = 0; q < 4; ++q) red[32 * q + warp] = sb[q];
    }
    __syncthreads();
    if (threadIdx.x < 4) {
        double t = 0.0;
        for (int w = 0; w < nwarp; ++w) t += red[32 * threadIdx.x + w];
        fp.SB[(4 * sb_sel + threadIdx.x) * FREE_SB_LD + blockIdx.x] = t;
    }
}

// The same with the per-source constants of this CTA's rows kept in shared memory for the whole solve (bie_gmres.cu): the
// tables are x_s times a constant of the geometry, so an application costs no global load besides x itself.
// K: shared, [3][rows2] double2: the (U, W) coefficients of class 0, of class 1, and (beta_0, beta_1)
//    (vortex-sheet matrix: (Er, Ei)/M_j, (M, 1)/M_j, unused).
__device__ __forceinline__ void free_init_row_consts(const NodeTable& nt, const CompTable& ct, const FreePlan& fp, int r0, int r1,
                                                     double2* K, int rows2)
{
    for (int s = r0 + threadIdx.x; s < r1; s += blockDim.x) {
        const double2 e = nt.E[s], q = nt.Q[s];
        const int l = s - r0;
        if (fp.vortex) {
            const double M = nt.MT[s].x;
            const int j = nt.COMP[s];
            const double m = 1.0 / (double)(ct.off[j + 1] - ct.off[j]);
            K[l] = make_double2(m * e.x, m * e.y);
            K[rows2 + l] = make_double2(m * M, m);
            K[2 * rows2 + l] = make_double2(0.0, 0.0);
            continue;
        }
        const bool src0 = (nt.COMP[s] == 0);
        double a0, b0, a1, b1;
        if (src0) { a0 = -2.0 * q.y; b0 = q.x;  a1 = 2.0 * q.x;  b1 = q.y; }   // K_00 ; -G_k0
        else      { a0 = -2.0 * q.x; b0 = -q.y; a1 = -2.0 * q.y; b1 = q.x; }   // G_0j ; K_kj
        K[l] = make_double2(fma(a0, e.y, 2.0 * b0 * e.x), fma(-a0, e.x, 2.0 * b0 * e.y));
        K[rows2 + l] = make_double2(fma(a1, e.y, 2.0 * b1 * e.x), fma(-a1, e.x, 2.0 * b1 * e.y));
        K[2 * rows2 + l] = make_double2(b0, b1);
    }
    __syncthreads();
}

__device__ __forceinline__ void free_write_tables_cached(const FreePlan& fp, int np, int r0, int r1, const double* v, const double2* K,
                                                         int rows2, double* red, int sb_sel = 0)
{
    double sb[4] = {0.0, 0.0, 0.0, 0.0};
    for (int s = r0 + threadIdx.x; s < r1; s += blockDim.x) {
        const int l = s - r0;
        const double x = v[l];
        const double2 k0 = K[l], k1 = K[rows2 + l], bb = K[2 * rows2 + l];
        fp.T[s]      = make_double2(x * k0.x, x * k0.y);
        fp.T[np + s] = make_double2(x * k1.x, x * k1.y);
        if (s >= fp.s_off) { sb[0] = fma(x, bb.x, sb[0]); sb[1] = fma(x, bb.y, sb[1]); }
        else               { sb[2] = fma(x, bb.x, sb[2]); sb[3] = fma(x, bb.y, sb[3]); }
    }
    if (fp.vortex) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
#pragma unroll
    for (int q = 0; q < 4; ++q) sb[q] = bie_warp_sum(sb[q]);
    __syncthreads();
    if (lane == 0) {
#pragma unroll
        for (int q = 0; q < 4; ++q) red[32 * q + warp] = sb[q];
    }
    __syncthreads();
    if (threadIdx.x < 4) {
        double t = 0.0;
        for (int w = 0; w < nwarp; ++w) t += red[32 * threadIdx.x + w];
        fp.SB[(4 * sb_sel + threadIdx.x) * FREE_SB_LD + blockIdx.x] = t;
    }
}

// ---- step 2: this CTA's slab of the (row block x source) list -> partial sums in fp.PB --------------------
// scratch: shared, free_scratch_doubles() doubles, 16-byte aligned.  All threads of the team must call.
// poll() is called by every warp after each chunk of 32 sources (the hybrid operator consumes tiles of its stored
// block there, bie_gemv.cuh).
// VORTEX: the matrix S of Eqs. (4.14) + (4.17) (bie_build.cu, "Vortex-sheet variant"), in the (X, Y) form: entry x_s = (A_t X' + B_t Y')/den with
// X' = Ei_t P_s - Er_t Q_s, Y' = R_s - M_t B_s from the class-independent tables (P,Q) = mu_s E_s, (R,B) = mu_s (M_s, 1), and the
// row's (A_t, B_t) = (2u_i, -u_r) / +-(2u_r, u_i), u_t = zeta'_t/2, which depend on whether the SOURCE lies on Gamma_0: the
// warp's source range is cut at M_0.  13 FP64-pipe instructions per pair.
__device__ __forceinline__ void free_cp_async16(void* dst_shared, const void* src_global, unsigned src_bytes)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst_shared);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" :: "r"(d), "l"(src_global), "r"(src_bytes) : "memory");
}

template <bool VORTEX, class Poll>
__device__ __forceinline__ void free_parts_impl(const NodeTable& nt, const CompTable& ct, const FreePlan& fp, double* scratch,
                                                const Team& team, const Poll& poll)
{
    const int lane = team.tid & 31, warp = team.warp;
    const int c = blockIdx.x;
    if (c >= fp.Geff) return;
    double* wsum = scratch;                                                       // [16][128]
    double2* stage = reinterpret_cast<double2*>(scratch + FREE_HEAD_DOUBLES + warp * 2 * fp.stage_buf);  // this warp's 2 buffers
    const int np = nt.npad;
    const double taubar = __ldg(fp.taubar);
    long long u0 = free_slab_start(fp, c);
    const long long u1 = free_slab_start(fp, c + 1);
    int b = free_list_block(fp, u0);
    while (u0 < u1) {
        const long long ub = free_list_start(fp, b);
        const long long ue = min(u1, free_list_start(fp, b + 1));
        const int sbase = b < fp.nb_below ? fp.s_off : 0;                        // first source of this block's list
        const int sa = sbase + 2 * (int)(u0 - ub), sb = sbase + 2 * (int)(ue - ub);  // sources [sa, sb) of row block b
        const int cls = b < fp.NB0 ? 0 : 1;
        const int row0 = free_block_row0(fp, b);
        const int rows = free_block_rows(fp, b, nt.n);
        // this lane's targets
        double ter[FREE_NT], tei[FREE_NT], tm[FREE_NT], acc[FREE_NT];
        int thi[FREE_NT];
#pragma unroll
        for (int i = 0; i < FREE_NT; ++i) {
            const int t = row0 + min(lane + 32 * i, rows - 1);  // inactive slots shadow the last row; result dropped
            const double2 e = nt.E[t];
            ter[i] = e.x; tei[i] = e.y; tm[i] = nt.MT[t].x; acc[i] = 0.0;
            thi[i] = __double2hiint(taubar * tm[i]);
        }
        double ca[2][FREE_NT], cb[2][FREE_NT];   // VORTEX: (A_t, B_t) for sources on Gamma_0 [0] and on solids [1]
        if (VORTEX) {
#pragma unroll
            for (int i = 0; i < FREE_NT; ++i) {
                const int t = row0 + min(lane + 32 * i, rows - 1);
                const int k = nt.COMP[t];
                const double Mk = (double)(ct.off[k + 1] - ct.off[k]);
                const double2 q = nt.Q[t];
                const double ur = q.x * Mk, ui = q.y * Mk;
                if (cls == 0) { ca[0][i] = 2.0 * ui; cb[0][i] = -ur; ca[1][i] = -2.0 * ur; cb[1][i] = -ui; }   // K+_00 ; -G+_j0
                else          { ca[0][i] = 2.0 * ur; cb[0][i] = ui;  ca[1][i] = 2.0 * ui;  cb[1][i] = -ur; }   // G+_0k ; K+_jk
            }
        }
        // this warp's share of the sources, in units of 2
        const int units = (sb - sa) >> 1;
        const int wa_all = sa + 2 * (int)((long long)units * warp / team.nwarp);
        const int wb_all = sa + 2 * (int)((long long)units * (warp + 1) / team.nwarp);
        const double2* TE = nt.E;
        const double2* TPQ = fp.T + (VORTEX ? (size_t)0 : (size_t)cls * np);   // Eq. (3.16): (U, W) of the rows' class
        const double2* TRB = fp.T + (size_t)np;                                 // VORTEX only
        for (int sgm = 0; sgm < (VORTEX ? 2 : 1); ++sgm) {
        // VORTEX: sources on Gamma_0 first, then the solids (different row coefficients); else the whole range at once
        const int wa = VORTEX ? (sgm == 0 ? wa_all : max(wa_all, fp.M0)) : wa_all;
        const int wb = VORTEX ? (sgm == 0 ? min(wb_all, fp.M0) : wb_all) : wb_all;
        // warp-private double buffer filled by cp.async (L2 only: the tables change between applications), zero-filled past wb
        auto issue = [&](int base_, int bufi) {
            const int s = base_ + lane;
            const bool ok = s < wb;
            const int sc = ok ? s : wa;
            const unsigned sz = ok ? 16u : 0u;
            double2* sg = stage + bufi * (fp.stage_buf >> 1);
            free_cp_async16(sg + lane, TE + sc, sz);
            free_cp_async16(sg + 32 + lane, TPQ + sc, sz);
            if (VORTEX) free_cp_async16(sg + 64 + lane, TRB + sc, sz);
            asm volatile("cp.async.commit_group;" ::: "memory");
        };
        int buf = 0;
        __syncwarp();
        if (wa < wb) issue(wa, 0);
        const int len = 32;
        for (int base = wa; base < wb; base += len, buf ^= 1) {
            const double2* sg = stage + buf * (fp.stage_buf >> 1);
            asm volatile("cp.async.wait_group 0;" ::: "memory");
            __syncwarp();                                   // chunk landed for all lanes; the other buffer is no longer read
            if (base + len < wb) issue(base + len, buf ^ 1);
            const int cnt = min(len, wb - base);   // even
#pragma unroll FREE_SRC_UNROLL
            for (int j = 0; j < cnt; ++j) {
                const double2 e = sg[j], pq = sg[32 + j];
                double2 rb;
                if (VORTEX) rb = sg[64 + j];
#pragma unroll
                for (int i = 0; i < FREE_NT; ++i) {
                    const double dr = e.x - ter[i], di = e.y - tei[i];
                    const double den = fma(dr, dr, di * di);
                    double val;
                    if (VORTEX) {
                        const double X = fma(tei[i], pq.x, -(ter[i] * pq.y));
                        const double Y = fma(-tm[i], rb.y, rb.x);
                        val = fma(cb[sgm][i], Y, ca[sgm][i] * X);
                    } else {
                        val = fma(pq.y, di, pq.x * dr);     // U_s dr + W_s di
                    }
                    const double r = bie_rcp3(den);
                    if (!(__double2hiint(den) < thi[i])) acc[i] = fma(val, r, acc[i]);
                }
            }
            poll();
        }
        }
        // the warp sums, added in fixed order
#pragma unroll
        for (int i = 0; i < FREE_NT; ++i) wsum[warp * FREE_ROWS + lane + 32 * i] = acc[i];
        team_sync(team);
        for (int r = team.tid; r < FREE_ROWS; r += team.nthr) {
            double s = 0.0;
            for (int w = 0; w < team.nwarp; ++w) s += wsum[w * FREE_ROWS + r];
            fp.PB[(size_t)(b + c) * FREE_ROWS + r] = s;
        }
        team_sync(team);
        u0 = ue;
        ++b;
    }
}

template <class Poll>
__device__ __forceinline__ void free_parts_sym(const NodeTable& nt, const FreePlan& fp, double* scratch, const Team& team,
                                               const Poll& poll);

template <class Poll>
__device__ __forceinline__ void free_parts(const NodeTable& nt, const CompTable& ct, const FreePlan& fp, double* scratch,
                                           const Team& team, const Poll& poll)
{
    if (fp.sym) free_parts_sym(nt, fp, scratch, team, poll);     // variants A/B; s_off = 0 or a row-block boundary
    else if (fp.vortex) free_parts_impl<true>(nt, ct, fp, scratch, team, poll);
    else free_parts_impl<false>(nt, ct, fp, scratch, team, poll);
}

// ---- step 3 (after a grid barrier): y_local[t - r0] = scale * (partials + near entries - constants - E_k term) ---------
// xsrc: the vector of step 1 (global, complete).  All threads of the CTA must call; ends with __syncthreads.
__device__ __forceinline__ void free_gather(const NodeTable& nt, const CompTable& ct, const FreePlan& fp, int r0, int r1,
                                            const double* __restrict__ xsrc, double scale, double* scratch,
                                            double* y_local, int sb_sel = 0)
{
    double* csum = scratch + FREE_WARPS * FREE_ROWS;  // [2][BIE_MAX_COMP]: component sums over s >= s_off, over all s
    double* sbs = csum + 2 * BIE_MAX_COMP;            // [4] constants (free_write_tables)
    double* wred = scratch;   // [2][32] (the warp-sum area is free again)
    // the E_k weights of the first two components this CTA's rows meet: loaded here, looked at only when the component sums are formed
    int ek0 = -1, ek1 = -1;
    for (int k = 0; k < ct.ncomp; ++k) {
        if (!(ct.off[k] < r1 && ct.off[k + 1] > r0)) continue;          // CTA-uniform
        if (ek0 < 0) ek0 = k; else if (ek1 < 0) ek1 = k;
    }
    const double em0 = (ek0 >= 0) ? nt.DG[ct.off[ek0]].y : 0.0;
    const double em1 = (ek1 >= 0) ? nt.DG[ct.off[ek1]].y : 0.0;
    // Everything below is a handful of dependent L2 round trips (about 0.7 us each).  The loads of the independent chains are
    // ISSUED first and consumed later, so that the chains overlap instead of queueing behind one another:
    //   A: CSR range of the CTA's rows -> near columns and values -> x at those columns        (3 round trips)
    //   B: reverse partials of the symmetric loops                                               (1-2)
    //   C: per-CTA partials of the constants sum beta x                                          (1)
    //   D: forward partials of the row                                                           (1)
    const int rows_ = r1 - r0, rows2_ = (rows_ + 1) & ~1;
    double* rpart = scratch + FREE_HEAD_DOUBLES;             // [4][rows2_] quarter sums of the reverse partials (staging area: free again)
    double* prod = rpart + 4 * rows2_;                        // products of the near entries with x
    const int prod_cap = FREE_WARPS * 2 * fp.stage_buf - 4 * rows2_;
    // A1
    const int pbeg = fp.near_ptr[8 * (size_t)r0], pend = fp.near_ptr[8 * (size_t)r1];
    // D (the thread's first row; a thread has more than one row only when n > 512 SMs' worth)
    const bool rowt = (int)threadIdx.x < rows_;
    int r_kpos = 0, r_off = 0, r_clo = 0, r_chi = -1;
    long long r_X0 = 0, r_X1 = 0;
    double pbv[4] = {0.0, 0.0, 0.0, 0.0};
    if (rowt) {
        const int t = r0 + threadIdx.x;
        int b;
        if (t < fp.M0) { b = t / FREE_ROWS; r_off = t - b * FREE_ROWS; }
        else { const int d = t - fp.M0; b = d / FREE_ROWS; r_off = d - b * FREE_ROWS; b += fp.NB0; }
        r_kpos = fp.sym ? __ldg(fp.sym_pos + b) : b;   // position of the block in the work list
        r_X0 = fp.sym ? __ldg(fp.sym_cum + r_kpos) : free_list_start(fp, b);
        r_X1 = fp.sym ? __ldg(fp.sym_cum + r_kpos + 1) : free_list_start(fp, b + 1);
        r_clo = max((int)(((r_X0 + 1) * fp.Geff + fp.U - 1) / fp.U) - 1, 0);
        r_chi = min((int)((r_X1 * fp.Geff + fp.U - 1) / fp.U) - 1, fp.Geff - 1);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int c = r_clo + q;
            if (c <= r_chi) {
                const long long a = max(free_slab_start(fp, c), r_X0), e = min(free_slab_start(fp, c + 1), r_X1);
                if (a < e) pbv[q] = __ldcg(fp.PB + (size_t)(r_kpos + c) * FREE_ROWS + r_off);
            }
        }
    }
    // B: symmetric work split, row t of block J also receives sum_{I < J} PC[I][t] (rows below s_off: nothing, their mirror
    // entries are stored).  Up to NB - 1 loads per row, each from another L2 line: four threads share a row (I = q, q + 4, ...;
    // sixteen loads in flight each); the four partial sums are added in fixed order by the row's thread.
    if (fp.sym) {
        for (int w = threadIdx.x; w < 4 * rows_; w += blockDim.x) {
            const int q = w / rows_, lr = w - q * rows_;
            const int t = r0 + lr;
            const int b = t < fp.s_off ? 0 : (t < fp.M0 ? t / FREE_ROWS : fp.NB0 + (t - fp.M0) / FREE_ROWS);
            const double* pc = fp.PC + t;
            double a0 = 0.0, a1 = 0.0;
            int I = q;
            for (; I + 60 < b; I += 64) {
                double v[16];
#pragma unroll
                for (int k = 0; k < 16; ++k) v[k] = __ldcg(pc + (size_t)(I + 4 * k) * nt.npad);
#pragma unroll
                for (int k = 0; k < 16; k += 2) { a0 += v[k]; a1 += v[k + 1]; }
            }
            for (; I + 28 < b; I += 32) {
                double v[8];
#pragma unroll
                for (int k = 0; k < 8; ++k) v[k] = __ldcg(pc + (size_t)(I + 4 * k) * nt.npad);
#pragma unroll
                for (int k = 0; k < 8; k += 2) { a0 += v[k]; a1 += v[k + 1]; }
            }
            for (; I < b; I += 4) a0 += __ldcg(pc + (size_t)I * nt.npad);
            rpart[q * rows2_ + lr] = a0 + a1;
        }
    }
    // A2, A3: the near entries of this CTA's rows are contiguous in the CSR arrays: all threads multiply them with x in
    // parallel, each row then adds its run from shared memory.  (Hybrid operator, or more entries than fit: every row walks
    // its own list below.)
    const bool flat = (fp.s_off == 0) && (pend - pbeg <= prod_cap);
    if (flat)
        for (int p = pbeg + threadIdx.x; p < pend; p += blockDim.x) prod[p - pbeg] = fp.near_val[p] * __ldcg(xsrc + fp.near_col[p]);
    // C: sum_s beta_s x_s per class and source range, the per-CTA partials of free_write_tables in fixed order (warps 0..3)
    if (!fp.vortex && threadIdx.x < 128) {
        const int q = threadIdx.x >> 5, lane = threadIdx.x & 31;
        double sb = 0.0;
        for (int i = lane; i < (int)gridDim.x; i += 32) sb += __ldcg(fp.SB + (4 * sb_sel + q) * FREE_SB_LD + i);
        sb = bie_warp_sum(sb);
        if (lane == 0) sbs[q] = sb;
    }
    // (the component sums come last, with the component's weight loaded at the top: stand-alone operator 0.1615 -> 0.158 ms at
    // config 5; the GMRES step did not change)
    {   // sum of x over each OBSTACLE component (em != 0) that owns one of this CTA's rows: all warps share the
        // component, lanes strided, warp sums added in fixed order -- every CTA gets the same bits.  Rows below s_off
        // (hybrid) only want the sources from s_off on, the stored block has the others.
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
        for (int k = 0; k < ct.ncomp; ++k) {
            if (!(ct.off[k] < r1 && ct.off[k + 1] > r0)) continue;      // CTA-uniform
            const double emk = (k == ek0) ? em0 : ((k == ek1) ? em1 : nt.DG[ct.off[k]].y);
            if (emk == 0.0) { if (threadIdx.x == 0) { csum[k] = 0.0; csum[BIE_MAX_COMP + k] = 0.0; } continue; }
            double shi = 0.0, slo = 0.0;
            for (int i = ct.off[k] + threadIdx.x; i < ct.off[k + 1]; i += blockDim.x) {
                const double xv = __ldcg(xsrc + i);
                if (i >= fp.s_off) shi += xv; else slo += xv;
            }
            shi = bie_warp_sum(shi); slo = bie_warp_sum(slo);
            if (lane == 0) { wred[warp] = shi; wred[32 + warp] = slo; }
            __syncthreads();
            if (threadIdx.x == 0) {
                double th = 0.0, tl = 0.0;
                for (int w = 0; w < nwarp; ++w) { th += wred[w]; tl += wred[32 + w]; }
                csum[k] = th;
                csum[BIE_MAX_COMP + k] = th + tl;
            }
            __syncthreads();
        }
    }
    __syncthreads();
    for (int t = r0 + threadIdx.x; t < r1; t += blockDim.x) {
        const int l = t - r0;
        double s;
        if (l == (int)threadIdx.x) {       // the row whose forward partials were loaded above
            s = (pbv[0] + pbv[1]) + (pbv[2] + pbv[3]);
            for (int c = r_clo + 4; c <= r_chi; ++c) {
                const long long a = max(free_slab_start(fp, c), r_X0), e = min(free_slab_start(fp, c + 1), r_X1);
                if (a < e) s += __ldcg(fp.PB + (size_t)(r_kpos + c) * FREE_ROWS + r_off);
            }
        } else {                            // more rows than threads
            int b, off;
            if (t < fp.M0) { b = t / FREE_ROWS; off = t - b * FREE_ROWS; }
            else { const int d = t - fp.M0; b = d / FREE_ROWS; off = d - b * FREE_ROWS; b += fp.NB0; }
            const int kpos = fp.sym ? __ldg(fp.sym_pos + b) : b;
            const long long X0 = fp.sym ? __ldg(fp.sym_cum + kpos) : free_list_start(fp, b);
            const long long X1 = fp.sym ? __ldg(fp.sym_cum + kpos + 1) : free_list_start(fp, b + 1);
            const int c_lo = max((int)(((X0 + 1) * fp.Geff + fp.U - 1) / fp.U) - 1, 0);
            const int c_hi = min((int)((X1 * fp.Geff + fp.U - 1) / fp.U) - 1, fp.Geff - 1);
            s = 0.0;
            for (int c = c_lo; c <= c_hi; ++c) {
                const long long a = max(free_slab_start(fp, c), X0), e = min(free_slab_start(fp, c + 1), X1);
                if (a < e) s += __ldcg(fp.PB + (size_t)(kpos + c) * FREE_ROWS + off);
            }
        }
        if (fp.sym) s += (rpart[l] + rpart[rows2_ + l]) + (rpart[2 * rows2_ + l] + rpart[3 * rows2_ + l]);
        // near pairs (rows below s_off: only the columns the stored block lacks)
        const bool below = (t < fp.s_off);
        const int p0 = fp.near_ptr[8 * (size_t)t], p1 = fp.near_ptr[8 * (size_t)t + 8];
        double sn = 0.0;
        if (flat) {
            for (int p = p0; p < p1; ++p) sn += prod[p - pbeg];
        } else {
            for (int p = p0; p < p1; ++p) {
                const int cix = fp.near_col[p];
                if (!below || cix >= fp.s_off) sn = fma(fp.near_val[p], __ldcg(xsrc + cix), sn);
            }
        }
        s += sn;
        if (!fp.vortex) {
            const int cl = t < fp.M0 ? 0 : 1;
            s -= below ? sbs[cl] : (sbs[cl] + sbs[2 + cl]);
        }
        const int k = nt.COMP[t];
        s = fma(-nt.DG[t].y, csum[(below ? 0 : BIE_MAX_COMP) + k], s);
        y_local[t - r0] = s * scale;
    }
    __syncthreads();
}

#include "bie_free_sym.cuh"   // free_parts_sym (declared above)
