// bie_free.cuh -- matrix-free form of SURVEY 8(a) row a6: y_t = sum_s A[t][s] x_s with the entries of
// Eq. (3.16) recomputed on the fly from the node tables; no matrix traffic at all.
// CTA-level device function shared by bie_matvec_free and the persistent GMRES kernel.
//
// Mapping.  A CTA owns the targets [r0, r1).  A thread keeps TWO targets in registers (their S, C, P, N and
// class) and runs over a share of the sources, which are staged tile by tile in shared memory and read as
// warp-wide broadcasts; the running sums stay in registers, so there is no reduction in the inner loop.
// The 512 threads form NG source groups of TG threads (TG = target slots, a power of two >= 32); group g
// takes the g-th part of every source tile; the NG partial sums per target are added in fixed order.
// The source's weight, the Re/Im selection of Eq. (3.10) and x_s are folded into two coefficient pairs per
// source, (u, v) x_s for targets on Gamma_0 and for targets on solids (see bie_build.cu for (u, v)).
// The rank-one E_k is applied as -(1/M_k) sum_{s in k} x_s after the pair loop.
#pragma once
#include "bie_common.cuh"

#define FREE_THREADS 512
#define FREE_TILE 512  // sources per shared-memory tile (one per thread)

__host__ __device__ inline int free_tg(int rows)
{
    int tg = 32;
    while (tg < FREE_THREADS && 2 * tg < rows) tg <<= 1;
    return tg;
}
// doubles of scratch: 2 tile buffers x 4 double2 arrays x FREE_TILE + group partials + component sums
__host__ __device__ inline int free_scratch_doubles(int rows_per_cta)
{
    return 2 * 8 * FREE_TILE + 2 * FREE_THREADS + BIE_MAX_COMP + 2;
}

struct FreeSrc {  // what one thread loads for one source of the next tile
    double S, C, P, N, qr, qi, x;
    int comp;
};

__device__ __forceinline__ FreeSrc free_load_src(const NodeTable& nt, const double* __restrict__ x, int s)
{
    FreeSrc f;
    if (s < nt.n) {
        f.S = nt.S[s]; f.C = nt.C[s]; f.P = nt.P[s]; f.N = nt.N[s];
        f.qr = nt.QR[s]; f.qi = nt.QI[s]; f.comp = nt.COMP[s];
        f.x = __ldcg(x + s);
    } else {  // beyond n: zero weight (contributes exactly 0, never near)
        f.S = 0.0; f.C = 1.0; f.P = 1.0e3; f.N = 1.0e-3; f.qr = 0.0; f.qi = 0.0; f.x = 0.0; f.comp = -1;
    }
    return f;
}

__device__ __forceinline__ void free_store_src(const FreeSrc& f, double2* buf, int i)
{
    const double ur = f.qr * f.x, ui = f.qi * f.x;
    buf[i] = make_double2(2.0 * f.S, 2.0 * f.C);
    buf[FREE_TILE + i] = make_double2(f.P, f.N);
    if (f.comp == 0) {
        buf[2 * FREE_TILE + i] = make_double2(ui, -ur);   // target on Gamma_0: Im c
        buf[3 * FREE_TILE + i] = make_double2(-ur, -ui);  // target on a solid: -Re c
    } else {
        buf[2 * FREE_TILE + i] = make_double2(ur, ui);    // target on Gamma_0: Re c
        buf[3 * FREE_TILE + i] = make_double2(ui, -ur);   // target on a solid: Im c
    }
}

struct FreeTgt {
    double S, C, P, N, acc;
    int idx, cls;  // cls: 0 target on Gamma_0, 1 on a solid
};

__device__ __forceinline__ void free_pair(FreeTgt& t, const double2 sc, const double2 pn, const double2 uv,
                                          const NodeTable& nt, const double* __restrict__ x, int sidx)
{
    const double sa = fma(sc.x, t.C, -(sc.y * t.S));
    const double ca = fma(sc.y, t.C, sc.x * t.S);
    const double ep = pn.x * t.N, en = pn.y * t.P;
    const double D = ep - en, G = ep + en;
    double nr = sa * ca, ni = D * G;
    const double den = fma(D, D, sa * sa);
    double r = bie_rcp(den);
    if (den < BIE_NEAR_TAU) {
        if (sidx == t.idx) {  // diagonal entry without its -E part (that is in the component sum)
            t.acc = fma(nt.DIAG[sidx] + nt.EM[sidx], __ldcg(x + sidx), t.acc);
            return;
        }
        double cr, ci;
        bie_cot_half_near(nt.X[sidx] - nt.X[t.idx], nt.Y[sidx] - nt.Y[t.idx], &cr, &ci);
        nr = cr; ni = -ci; r = 1.0;
    }
    t.acc = fma(fma(uv.y, ni, uv.x * nr), r, t.acc);
}

// y_local[t - r0] = sum_s A[t][s] x[s], t in [r0, r1).  x: global (read through L2).  scratch: shared,
// free_scratch_doubles() doubles, 16-byte aligned.  blockDim.x must be FREE_THREADS; r1 - r0 <= 2*FREE_THREADS.
__device__ __forceinline__ void bie_cta_matvec_free(const NodeTable& nt, const CompTable& ct, int r0, int r1,
                                                    const double* __restrict__ x, double* scratch, double* y_local)
{
    const int n = nt.n;
    const int rows = r1 - r0;
    const int TG = free_tg(rows), NG = FREE_THREADS / TG;
    const int slot = threadIdx.x & (TG - 1), grp = threadIdx.x / TG;
    double2* tile[2] = {reinterpret_cast<double2*>(scratch), reinterpret_cast<double2*>(scratch) + 4 * FREE_TILE};
    double* gpart = scratch + 2 * 8 * FREE_TILE;  // [2][FREE_THREADS]
    double* csum = gpart + 2 * FREE_THREADS;      // [ncomp]

    // component sums of x for the E_k term (fixed order: one warp per component, lanes strided)
    {
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
        for (int k = warp; k < ct.ncomp; k += FREE_THREADS / 32) {
            double s = 0.0;
            for (int i = ct.off[k] + lane; i < ct.off[k + 1]; i += 32) s += __ldcg(x + i);
            s = bie_warp_sum(s);
            if (lane == 0) csum[k] = s;
        }
    }
    FreeTgt tg[2];
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        const int loc = slot + q * TG;
        const int i = r0 + min(loc, rows - 1);  // inactive slots shadow the last target; result dropped
        tg[q].S = nt.S[i]; tg[q].C = nt.C[i]; tg[q].P = nt.P[i]; tg[q].N = nt.N[i];
        tg[q].acc = 0.0; tg[q].idx = i; tg[q].cls = (nt.COMP[i] == 0) ? 0 : 1;
    }
    const int per = FREE_TILE / NG;  // sources of a tile per group
    const int ntile = (n + FREE_TILE - 1) / FREE_TILE;
    FreeSrc nxt = free_load_src(nt, x, threadIdx.x);
    free_store_src(nxt, tile[0], threadIdx.x);
    __syncthreads();
    for (int it = 0; it < ntile; ++it) {
        const double2* cur = tile[it & 1];
        if (it + 1 < ntile) nxt = free_load_src(nt, x, (it + 1) * FREE_TILE + threadIdx.x);
        const double2* uv0 = cur + (2 + tg[0].cls) * FREE_TILE;
        const double2* uv1 = cur + (2 + tg[1].cls) * FREE_TILE;
        const int sb = grp * per;
#pragma unroll 2
        for (int j = sb; j < sb + per; ++j) {
            const double2 sc = cur[j], pn = cur[FREE_TILE + j];
            const int sidx = it * FREE_TILE + j;
            free_pair(tg[0], sc, pn, uv0[j], nt, x, sidx);
            free_pair(tg[1], sc, pn, uv1[j], nt, x, sidx);
        }
        if (it + 1 < ntile) free_store_src(nxt, tile[(it + 1) & 1], threadIdx.x);
        __syncthreads();
    }
    // sum the NG group partials per target in fixed order, then the E_k term
#pragma unroll
    for (int q = 0; q < 2; ++q) gpart[q * FREE_THREADS + threadIdx.x] = tg[q].acc;
    __syncthreads();
    for (int loc = threadIdx.x; loc < rows; loc += FREE_THREADS) {
        const int q = loc / TG, sl = loc - q * TG;
        double s = 0.0;
        for (int g = 0; g < NG; ++g) s += gpart[q * FREE_THREADS + g * TG + sl];
        const int t = r0 + loc;
        const int k = nt.COMP[t];
        s = fma(-nt.EM[t], csum[k], s);
        y_local[loc] = s;
    }
    __syncthreads();
}
