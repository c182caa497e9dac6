// bie_free.cuh -- matrix-free form of SURVEY 8(a) row a6: y_t = sum_s A[t][s] x_s with the entries of
// Eq. (3.16) recomputed on the fly from the node tables; no matrix traffic at all.
// Device functions for a TEAM of warps of one CTA (all of it in bie_matvec_free and in the matrix-free GMRES;
// half of it in the hybrid GMRES, where the other half streams stored columns from HBM).
//
// Mapping.  The CTA owns the targets [r0, r1).  A thread keeps TWO targets in registers (E_t, M_t and class) and
// runs over a share of the sources, which are staged tile by tile in shared memory and read as warp-wide
// broadcasts; the running sums stay in registers, so there is no reduction in the inner loop.  The team's
// threads form NG source groups of TG threads (TG = target slots / 2, a power of two >= 32); group g takes the
// g-th part of every source tile; the NG partial sums per target are added in fixed order at the end.
// The source's weight, the Re/Im selection of Eq. (3.10) and x_s are folded into two coefficient pairs per
// source, (alpha, beta) x_s for targets on Gamma_0 and for targets on solids (see bie_common.cuh).
// Per pair: 13 FP64-pipe instructions.  The inner loop is branch-free: near pairs (den < thr_s, including
// s == t) are left out by predication and only flagged; after every FREE_SB sources the warp votes and, if
// needed, revisits those sources for the near pairs alone (Laurent series / diagonal limit).
// The rank-one E_k is applied as -(1/M_k) sum_{s in k} x_s after the pair loop.
#pragma once
#include "bie_common.cuh"

#define FREE_THREADS 512
#define FREE_SB 32   // sources between near votes

struct FreeTeam {
    int tid;   // 0 .. nthr-1
    int nthr;  // multiple of 32; source tile = nthr sources (one per thread)
    int bar;   // named barrier id used by this team (0 = the whole CTA)
};
__device__ __forceinline__ void team_sync(const FreeTeam& tm)
{
    asm volatile("bar.sync %0, %1;" ::"r"(tm.bar), "r"(tm.nthr) : "memory");
}

__host__ __device__ inline int free_tg(int rows, int nthr)
{
    int tg = 32;
    while (tg < nthr && 2 * tg < rows) tg <<= 1;
    return tg;
}
// doubles of scratch for a team of nthr threads: 2 tile buffers x 4 double2 arrays x nthr, group partials
// [2][nthr], component sums
__host__ __device__ inline int free_scratch_doubles(int nthr) { return 2 * 8 * nthr + 2 * nthr + BIE_MAX_COMP + 2; }

struct FreeSrc {  // what one thread loads for one source of the next tile
    double2 e, mt, q;
    double x;
    int comp;
};

__device__ __forceinline__ FreeSrc free_load_src(const NodeTable& nt, const double* __restrict__ x, double scale,
                                                 int s, int s_end)
{
    FreeSrc f;
    if (s < s_end) {
        f.e = nt.E[s]; f.mt = nt.MT[s]; f.q = nt.Q[s]; f.comp = nt.COMP[s];
        f.x = __ldcg(x + s) * scale;
    } else {  // beyond the range: zero weight (contributes exactly 0), never near (thr = 0)
        f.e = make_double2(0.0, 0.0); f.mt = make_double2(0.0, 0.0); f.q = make_double2(0.0, 0.0);
        f.x = 0.0; f.comp = -1;
    }
    return f;
}

__device__ __forceinline__ void free_store_src(const FreeSrc& f, double2* buf, int nthr, int i)
{
    const double ur = f.q.x * f.x, ui = f.q.y * f.x;
    buf[i] = f.e;
    buf[nthr + i] = f.mt;
    if (f.comp == 0) {
        buf[2 * nthr + i] = make_double2(-2.0 * ui, ur);   // target on Gamma_0: Im c
        buf[3 * nthr + i] = make_double2(2.0 * ur, ui);    // target on a solid: -Re c
    } else {
        buf[2 * nthr + i] = make_double2(-2.0 * ur, -ui);  // target on Gamma_0: Re c
        buf[3 * nthr + i] = make_double2(-2.0 * ui, ur);   // target on a solid: Im c
    }
}

struct FreeState {
    double er[2], ei[2], m[2], acc[2];
    int idx[2], cls[2];  // cls: 0 target on Gamma_0, 1 on a solid
    int TG, NG, slot, grp;
};

__device__ __forceinline__ void free_begin(FreeState& st, const NodeTable& nt, int r0, int r1, const FreeTeam& tm)
{
    const int rows = r1 - r0;
    st.TG = free_tg(rows, tm.nthr);
    st.NG = tm.nthr / st.TG;
    st.slot = tm.tid & (st.TG - 1);
    st.grp = tm.tid / st.TG;
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        const int loc = st.slot + q * st.TG;
        const int i = r0 + min(loc, rows - 1);  // inactive slots shadow the last target; result dropped
        const double2 e = nt.E[i];
        st.er[q] = e.x; st.ei[q] = e.y; st.m[q] = nt.MT[i].x;
        st.acc[q] = 0.0; st.idx[q] = i; st.cls[q] = (nt.COMP[i] == 0) ? 0 : 1;
    }
}

// near pairs of the sources [jb, je) of the current tile, for one thread's two targets (rare path): returns the
// two sums of their exact contributions.  Everything by value, so that the caller's state stays in registers.
static __device__ __noinline__ double2 free_near_fix(const double2* __restrict__ DG, const double2* __restrict__ XY,
                                                     const double* __restrict__ x, double scale, const double2* cur,
                                                     int nthr, int jb, int je, int sbase, double er0, double ei0,
                                                     double er1, double ei1, int idx0, int idx1, int cls0, int cls1)
{
    double add[2] = {0.0, 0.0};
    const double ter[2] = {er0, er1}, tei[2] = {ei0, ei1};
    const int tidx[2] = {idx0, idx1}, tcls[2] = {cls0, cls1};
    for (int j = jb; j < je; ++j) {
        const double2 e = cur[j];
        const int thi = __double2hiint(cur[nthr + j].y);
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            const double dr = e.x - ter[q], di = e.y - tei[q];
            const double den = fma(dr, dr, di * di);
            if (__double2hiint(den) < thi) {
                const int sidx = sbase + j;
                if (sidx == tidx[q]) {  // diagonal entry without its -E part (that is in the component sum)
                    const double2 dg = DG[sidx];
                    add[q] = fma(dg.x + dg.y, __ldcg(x + sidx) * scale, add[q]);
                } else {
                    const double2 zs = XY[sidx], zt = XY[tidx[q]];
                    double cr, ci;
                    bie_cot_half_near(zs.x - zt.x, zs.y - zt.y, &cr, &ci);
                    const double2 ab = cur[(2 + tcls[q]) * nthr + j];
                    add[q] += fma(ab.y, ci, -0.5 * ab.x * cr);
                }
            }
        }
    }
    return make_double2(add[0], add[1]);
}

// adds the contribution of the sources [c_lo, c_hi) (x scaled by `scale`) to the running sums.
// scratch: shared, free_scratch_doubles(nthr) doubles, 16-byte aligned.  All threads of the team must call.
__device__ __forceinline__ void free_chunk(FreeState& st, const NodeTable& nt, int c_lo, int c_hi,
                                           const double* __restrict__ x, double scale, double* scratch,
                                           const FreeTeam& tm)
{
    const int nthr = tm.nthr;
    double2* const tile0 = reinterpret_cast<double2*>(scratch);  // two buffers of 4 nthr double2 each
    const int per = nthr / st.NG;  // sources of a tile per group (= TG >= 32, a multiple of FREE_SB)
    const int ntile = (c_hi - c_lo + nthr - 1) / nthr;
    if (ntile <= 0) return;
    FreeSrc nxt = free_load_src(nt, x, scale, c_lo + tm.tid, c_hi);
    team_sync(tm);  // previous users of the tile buffers are done
    free_store_src(nxt, tile0, nthr, tm.tid);
    team_sync(tm);
    const unsigned thr_lane_any = 0xffffffffu;
    for (int it = 0; it < ntile; ++it) {
        const double2* cur = tile0 + (it & 1) * 4 * nthr;
        if (it + 1 < ntile) nxt = free_load_src(nt, x, scale, c_lo + (it + 1) * nthr + tm.tid, c_hi);
        const double2* sE = cur;
        const double2* sMT = cur + nthr;
        const double2* ab0 = cur + (2 + st.cls[0]) * nthr;
        const double2* ab1 = cur + (2 + st.cls[1]) * nthr;
        const int sb = st.grp * per;
        for (int jb = sb; jb < sb + per; jb += FREE_SB) {
            int flag = 0;
#pragma unroll 2
            for (int j = jb; j < jb + FREE_SB; ++j) {
                const double2 e = sE[j], mt = sMT[j];
                const int thi = __double2hiint(mt.y);
                {
                    const double2 ab = ab0[j];
                    const double dr = e.x - st.er[0], di = e.y - st.ei[0];
                    const double den = fma(dr, dr, di * di);
                    const double X = fma(st.ei[0], e.x, -(st.er[0] * e.y));
                    const double Y = mt.x - st.m[0];
                    const double val = fma(ab.y, Y, ab.x * X);
                    const double r = bie_rcp3(den);
                    const bool near = __double2hiint(den) < thi;
                    flag |= near ? 1 : 0;
                    if (!near) st.acc[0] = fma(val, r, st.acc[0]);
                }
                {
                    const double2 ab = ab1[j];
                    const double dr = e.x - st.er[1], di = e.y - st.ei[1];
                    const double den = fma(dr, dr, di * di);
                    const double X = fma(st.ei[1], e.x, -(st.er[1] * e.y));
                    const double Y = mt.x - st.m[1];
                    const double val = fma(ab.y, Y, ab.x * X);
                    const double r = bie_rcp3(den);
                    const bool near = __double2hiint(den) < thi;
                    flag |= near ? 1 : 0;
                    if (!near) st.acc[1] = fma(val, r, st.acc[1]);
                }
            }
            if (__any_sync(thr_lane_any, flag)) {
                if (flag) {
                    const double2 d = free_near_fix(nt.DG, nt.XY, x, scale, cur, nthr, jb, jb + FREE_SB, c_lo + it * nthr,
                                                    st.er[0], st.ei[0], st.er[1], st.ei[1], st.idx[0], st.idx[1],
                                                    st.cls[0], st.cls[1]);
                    st.acc[0] += d.x; st.acc[1] += d.y;
                }
            }
        }
        if (it + 1 < ntile) free_store_src(nxt, tile0 + ((it + 1) & 1) * 4 * nthr, nthr, tm.tid);
        team_sync(tm);
    }
}

// y_local[t - r0] = running sums + E_k term over the sources [c_lo, c_hi) that were processed.
// All threads of the team must call; ends with a team_sync.
__device__ __forceinline__ void free_end(FreeState& st, const NodeTable& nt, const CompTable& ct, int r0, int r1,
                                         int c_lo, int c_hi, const double* __restrict__ x, double scale,
                                         double* scratch, double* y_local, bool accumulate, const FreeTeam& tm)
{
    const int nthr = tm.nthr;
    const int rows = r1 - r0;
    double* gpart = scratch + 2 * 8 * nthr;  // [2][nthr]
    double* csum = gpart + 2 * nthr;         // [ncomp]
    // component sums of x over the processed range (fixed order: one warp per component, lanes strided)
    {
        const int lane = tm.tid & 31, warp = tm.tid >> 5;
        for (int k = warp; k < ct.ncomp; k += nthr / 32) {
            const int a = max(ct.off[k], c_lo), b = min(ct.off[k + 1], c_hi);
            double s = 0.0;
            for (int i = a + lane; i < b; i += 32) s += __ldcg(x + i);
            s = bie_warp_sum(s);
            if (lane == 0) csum[k] = s * scale;
        }
    }
#pragma unroll
    for (int q = 0; q < 2; ++q) gpart[q * nthr + tm.tid] = st.acc[q];
    team_sync(tm);
    for (int loc = tm.tid; loc < rows; loc += nthr) {
        const int q = loc / st.TG, sl = loc - q * st.TG;
        double s = 0.0;
        for (int g = 0; g < st.NG; ++g) s += gpart[q * nthr + g * st.TG + sl];
        const int t = r0 + loc;
        const int k = nt.COMP[t];
        s = fma(-nt.DG[t].y, csum[k], s);
        y_local[loc] = accumulate ? y_local[loc] + s : s;
    }
    team_sync(tm);
}

// whole operator for a CTA (team = all threads): y_local[t - r0] = sum_s A[t][s] (scale x[s]), t in [r0, r1)
__device__ __forceinline__ void bie_cta_matvec_free(const NodeTable& nt, const CompTable& ct, int r0, int r1,
                                                    const double* __restrict__ x, double scale, double* scratch,
                                                    double* y_local)
{
    FreeTeam tm;
    tm.tid = threadIdx.x; tm.nthr = blockDim.x; tm.bar = 0;
    FreeState st;
    free_begin(st, nt, r0, r1, tm);
    free_chunk(st, nt, 0, nt.n, x, scale, scratch, tm);
    free_end(st, nt, ct, r0, r1, 0, nt.n, x, scale, scratch, y_local, false, tm);
}
