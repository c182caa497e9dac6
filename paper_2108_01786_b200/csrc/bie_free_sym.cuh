// bie_free_sym.cuh -- the matrix-free operator of bie_free.cuh using the ODDNESS of the kernel:
//     cot((zeta_s - zeta_t)/2) = -cot((zeta_t - zeta_s)/2),
// so den = |E_s - E_t|^2, its reciprocal and the differences E_s - E_t serve the entry (t,s) AND the entry (s,t) of
// Eq. (3.16) (SURVEY section 7 "oddness").  Per pair of entries, in the difference form of bie_common.cuh: 2 sub + 2 den + 3 rcp
// shared, 2 + 1 for each direction (forward (U_s dr + W_s di)/den, reverse -(U'_t dr + W'_t di)/den: E_t - E_s = -(dr + i di)):
// 13 FP64-pipe instructions for two entries instead of 20, plus the lane reduction of the reverse sums.
//
// Work split.  Row block I (FREE_ROWS rows of one class) x the sources s >= row0(I): the block's own rows one-directionally
// (all their pairs are inside), the later sources symmetrically -- forward A[t][s] x_s into the lane's register sums as in
// bie_free.cuh, reverse A[s][t] x_t summed over the 128 targets of the block into a per-(row block, source) partial
// PC[I][s] in L2.  The triangular list is cut into equal slabs of sources, one per CTA.  The owner of row t (block J)
// gathers the forward partials of J and  sum_{I < J} PC[I][t]  in fixed order: deterministic.
// Reverse sums of 8 consecutive sources are reduced over the lanes through lane-private shared-memory slots (a transposing
// shuffle butterfly was 3 % slower: its 9 dependent steps stall the warp).
// Near pairs.  In the block's own rows (which hold the pair s == t, den = 0) a pair with den < taubar M_t is left out by
// predication, as in bie_free.cuh.  In the symmetric segments there is NO test at all: every pair is summed with the fast
// arithmetic, and the CSR near matrix of bie_near.cu stores, for the pairs it lists that lie in different row blocks,
// the CORRECTION exact - fast instead of the exact entry.  Both fast values come from the same rounded E_s - E_t, so they
// agree to a few ulp and the correction is as accurate as the exact entry; the pair loop loses two compares and four
// selects per pair and the registers of the thresholds (ncu: the loop was bound by issue slots and latency, not by
// the FP64 pipe).  Distinct nodes that coincide exactly (a pole of the kernel) give Inf/NaN, as the exact entry would.
// Hybrid operator (fp.s_off > 0, a row-block boundary): the leading s_off x s_off block is stored; every other pair {t, s},
// t < s, has s >= s_off, so the list is the same triangle with the sources cut at s_off: row blocks below s_off take the
// sources [s_off, npad) symmetrically (forward into their rows, reverse into the rows from s_off on).
#pragma once
#include "bie_free.cuh"

// The triangular list is laid out in the order perm[0], perm[1], ... = 0, NB-1, 1, NB-2, ... (long and short source lists
// alternate, so that every CTA's slab holds one or two long parts and at most a few short ones); cum[k] = sources before
// position k.  Tables in device memory (FreePlan::sym_cum / sym_perm / sym_pos, bie_nodes.cu).
__device__ __forceinline__ int sym_find_pos(const FreePlan& fp, long long u)
{
    int lo = 0, hi = fp.NB - 1;   // largest k with cum[k] <= u
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (__ldg(fp.sym_cum + mid) <= u) lo = mid; else hi = mid - 1;
    }
    return lo;
}

// this CTA's slab of the triangular (row block x later sources) list -> forward partials in fp.PB, reverse partials in fp.PC.
// scratch: shared, free_scratch_doubles(false, true) doubles.  All threads of the team must call.  poll(): see free_parts_impl.
template <class Poll>
__device__ __forceinline__ void free_parts_sym(const NodeTable& nt, const FreePlan& fp, double* scratch, const Team& team,
                                               const Poll& poll)
{
    const int lane = team.tid & 31, warp = team.warp, nwarp = team.nwarp;
    const int c = blockIdx.x;
    if (c >= fp.Geff) return;
    double* wsum = scratch;
    const int sbuf = fp.stage_buf;                                   // 128 doubles: E [32] double2, (U,W) [32] double2
    double* stage = scratch + FREE_HEAD_DOUBLES + warp * 2 * sbuf;
    double* col = scratch + FREE_HEAD_DOUBLES + FREE_WARPS * 2 * sbuf + warp * (SYM_BATCH * SYM_COL_STRIDE);   // this warp's reverse sums of a batch
    const int np = nt.npad;
    const double taubar = __ldg(fp.taubar);
    long long u0 = (long long)c * fp.U / fp.Geff;
    const long long u1 = (long long)(c + 1) * fp.U / fp.Geff;
    int k = sym_find_pos(fp, u0);
    const double2 zero2 = make_double2(0.0, 0.0);
    while (u0 < u1) {
        const int b = __ldg(fp.sym_perm + k);
        const long long ub = __ldg(fp.sym_cum + k);
        const long long ue = min(u1, __ldg(fp.sym_cum + k + 1));
        const int cls = b < fp.NB0 ? 0 : 1;
        const int row0 = free_block_row0(fp, b);
        const int rows = free_block_rows(fp, b, nt.n);
        const bool below = (row0 + rows <= fp.s_off);        // hybrid: a row block of the stored block's rows
        const int src0 = below ? fp.s_off : row0;
        // list positions [ub, ub + SYM_PART_PAD) of a block are virtual (bie_free.cuh): sources [sa, sb), all >= src0
        const int sa = src0 + (int)max(0LL, (u0 - ub) - SYM_PART_PAD), sb = src0 + (int)max(0LL, (ue - ub) - SYM_PART_PAD);
        double ter[FREE_NT], tei[FREE_NT], acc[FREE_NT];
        int thi[FREE_NT];
        bool live[FREE_NT];
#pragma unroll
        for (int i = 0; i < FREE_NT; ++i) {
            live[i] = (lane + 32 * i < rows);
            const int t = row0 + min(lane + 32 * i, rows - 1);   // inactive slots shadow the last row; forward result dropped
            const double2 e = nt.E[t];
            ter[i] = e.x; tei[i] = e.y; acc[i] = 0.0;
            thi[i] = __double2hiint(taubar * nt.MT[t].x);
        }
        const int span = sb - sa;
        const int wa_all = sa + (int)((long long)span * warp / nwarp);
        const int wb_all = sa + (int)((long long)span * (warp + 1) / nwarp);
        const int d_end = below ? src0 : row0 + rows;         // end of the one-directional sources (the block's own rows)
        const int c_end = (cls == 0) ? max(fp.M0, src0) : np; // end of the sources of the block's own class
        const double2* TUW = fp.T + (size_t)cls * np;            // forward tables: (U, W) for the class of the block's rows
        for (int sgm = 0; sgm < 3; ++sgm) {
            // 0: own rows (one direction); 1: later sources of the same class; 2: sources on solids below a Gamma_0 block
            const int lo = sgm == 0 ? src0 : (sgm == 1 ? d_end : c_end);
            const int hi = sgm == 0 ? d_end : (sgm == 1 ? c_end : np);
            const int wa = max(wa_all, lo), wb = min(wb_all, hi);
            if (wa >= wb) continue;                          // warp-uniform
            const bool rev = (sgm != 0);
            const int rcls = (sgm == 2) ? 1 : cls;           // class of the ROWS of the reverse entries (= of these sources)
            double tu[FREE_NT], tw[FREE_NT];
#pragma unroll
            for (int i = 0; i < FREE_NT; ++i) {
                tu[i] = tw[i] = 0.0;
                if (rev && live[i]) {                        // this target as a SOURCE of rows of class rcls
                    const int t = row0 + lane + 32 * i;
                    const double2 uw = __ldcg(fp.T + (size_t)rcls * np + t);
                    tu[i] = uw.x; tw[i] = uw.y;
                }
            }
            // warp-private double buffer filled by cp.async (no registers held across a chunk), zero-filled past wb: the batches
            // run over multiples of SYM_BATCH and the sources beyond wb must be zero sources
            auto issue = [&](int base_, int bufi) {
                const int s = base_ + lane;
                const bool ok = s < wb;
                const int sc = ok ? s : wa;
                const unsigned sz = ok ? 16u : 0u;
                double2* sgi = reinterpret_cast<double2*>(stage + bufi * sbuf);
                free_cp_async16(sgi + lane, nt.E + sc, sz);
                free_cp_async16(sgi + 32 + lane, TUW + sc, sz);
                asm volatile("cp.async.commit_group;" ::: "memory");
            };
            int buf = 0;
            __syncwarp();
            issue(wa, 0);
            const int len = 32;
            for (int base = wa; base < wb; base += len, buf ^= 1) {
                const double2* sg = reinterpret_cast<const double2*>(stage + buf * sbuf);
                asm volatile("cp.async.wait_group 0;" ::: "memory");
                __syncwarp();                                   // chunk landed for all lanes; the other buffer is no longer read
                if (base + len < wb) issue(base + len, buf ^ 1);
                const int cnt = min(len, wb - base);
                if (!rev) {
#pragma unroll 2
                    for (int j = 0; j < cnt; ++j) {
                        const double2 e = sg[j], uw = sg[32 + j];
#pragma unroll
                        for (int i = 0; i < FREE_NT; ++i) {
                            const double dr = e.x - ter[i], di = e.y - tei[i];
                            const double den = fma(dr, dr, di * di);
                            const double val = fma(uw.y, di, uw.x * dr);
                            const double r = bie_rcp3(den);
                            if (!(__double2hiint(den) < thi[i])) acc[i] = fma(val, r, acc[i]);
                        }
                    }
                } else {
                    for (int j0 = 0; j0 < cnt; j0 += SYM_BATCH) {   // sources beyond cnt are zero sources; not written
                        // the next source's operands are loaded BEFORE this source's reverse sum is stored: the compiler
                        // cannot move a shared load above a shared store it cannot tell apart, and would serialise the sources
                        double2 e = sg[j0], uw = sg[32 + j0];
#pragma unroll
                        for (int u = 0; u < SYM_BATCH; ++u) {
                            const int j = j0 + u;
                            double2 en = e, uwn = uw;
                            if (u + 1 < SYM_BATCH) { en = sg[j + 1]; uwn = sg[32 + j + 1]; }
                            double s_rev0 = 0.0, s_rev1 = 0.0;
#pragma unroll
                            for (int i = 0; i < FREE_NT; ++i) {
                                const double dr = e.x - ter[i], di = e.y - tei[i];
                                const double den = fma(dr, dr, di * di);
                                const double val = fma(uw.y, di, uw.x * dr);
                                const double r = bie_rcp3(den);
                                acc[i] = fma(val, r, acc[i]);
                                // reverse entry A[s][t] x_t: row s, source t (its (U, W) for the class of s), E_t - E_s = -(dr + i di);
                                // the sign is applied once, after the lane reduction
                                const double vr = fma(tw[i], di, tu[i] * dr);
                                if (i & 1) s_rev1 = fma(vr, r, s_rev1); else s_rev0 = fma(vr, r, s_rev0);
                            }
                            e = en; uw = uwn;
                            col[u * SYM_COL_STRIDE + lane] = s_rev0 + s_rev1;
                        }
                        // lane reduction of the SYM_BATCH reverse sums through shared memory: 32 / SYM_BATCH lanes share a source,
                        // each adds 8 slots, shuffles finish (fixed order)
                        __syncwarp();
                        {
                            constexpr int LPS = 32 / SYM_BATCH;                 // lanes per source (4 for a batch of 8)
                            constexpr int SPL = 32 / LPS;                        // slots per lane (8)
                            const double* cp = col + (lane / LPS) * SYM_COL_STRIDE + SPL * (lane % LPS);
                            double v = 0.0;
#pragma unroll
                            for (int q = 0; q < SPL; q += 2) v += cp[q] + cp[q + 1];
#pragma unroll
                            for (int o = LPS >> 1; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                            const int j = j0 + lane / LPS;
                            if ((lane % LPS) == 0 && j < cnt) fp.PC[(size_t)b * np + base + j] = -v;
                        }
                        __syncwarp();
                    }
                }
                poll();
            }
        }
        // the warp sums of the forward direction, added in fixed order
#pragma unroll
        for (int i = 0; i < FREE_NT; ++i) wsum[warp * FREE_ROWS + lane + 32 * i] = acc[i];
        team_sync(team);
        for (int r = team.tid; r < FREE_ROWS; r += team.nthr) {
            double s = 0.0;
            for (int w = 0; w < nwarp; ++w) s += wsum[w * FREE_ROWS + r];
            fp.PB[(size_t)(k + c) * FREE_ROWS + r] = s;
        }
        team_sync(team);
        u0 = ue;
        ++k;
    }
}
