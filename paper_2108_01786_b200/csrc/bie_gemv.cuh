// bie_gemv.cuh -- SURVEY 8(a) row a6: the dense FP64 GEMV y = A x of the Krylov matvec (PAPER.md:L857,
// "level 2 BLAS speed" PAPER.md:L921), as a CTA-level device function shared by bie_matvec and by the
// persistent GMRES kernel.  HBM-bound: 8 B read per entry, 2 flops.
//
// A CTA owns a contiguous block of rows [r0, r1).  Work is cut into units of (row pair) x (column chunk
// of gemv_chunk() doubles); the CTA's warps take units round-robin, so every warp has the same number of
// 128-bit loads to issue however the rows divide.  A warp streams its two rows with 2 x GEMV_UNROLL
// independent LDG.128 per lane in flight (512 contiguous bytes per warp-load), multiplies by x from shared
// memory (or from L2 when n is too large for shared memory), reduces by warp shuffles and leaves the
// partial sum in shared memory; partials are then summed over chunks in fixed order (deterministic).
#pragma once
#include "bie_common.cuh"

#define GEMV_UNROLL 4

// doubles per (row, chunk) unit: 2048 (32 warp-loads of 64 doubles) for large n; smaller for small n so
// that every warp of the CTA still gets a unit.  Always a multiple of 64.
__host__ __device__ inline int gemv_chunk(int rows_per_cta, int n, int nwarp)
{
    int chunk = 2048;
    const int npair = (rows_per_cta + 1) >> 1;
    while (chunk > 128 && npair * ((n + chunk - 1) / chunk) < 2 * nwarp) chunk >>= 1;
    // equal chunks: a short last chunk would always land on the same warps (units go round-robin)
    const int nch = (n + chunk - 1) / chunk;
    chunk = ((n + nch - 1) / nch + 63) & ~63;
    return chunk;
}

// streaming (evict-first) 128-bit load for matrices larger than L2; plain read-only load otherwise
template <bool STREAM>
__device__ __forceinline__ double2 gemv_ld(const double2* p)
{
    if (STREAM) return __ldcs(p);
    return __ldg(p);
}

// number of doubles of shared memory bie_cta_gemv needs for partial sums
__host__ __device__ inline int gemv_part_doubles(int rows_per_cta, int n, int chunk)
{
    const int nch = (n + chunk - 1) / chunk;
    return nch * ((rows_per_cta + 1) & ~1);
}

// y_local[r - r0] = sum_c A[r][c] * x[c] for r in [r0, r1).  xs: x in shared memory (XS = true) or global.
// part: shared scratch of gemv_part_doubles() doubles.  All threads of the team must call; ends with the
// results in y_local (shared) after a team barrier.  n = number of columns used (the hybrid operator passes
// the width of its stored slab).
// 128-bit load with an L2 eviction-priority hint (policy from createpolicy): the resident part of a streamed matrix
__device__ __forceinline__ double2 gemv_ld_hint(const double2* p, unsigned long long pol)
{
    double2 v;
    asm volatile("ld.global.nc.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol));
    return v;
}

// one (row pair) x (column chunk) unit of a warp: acc0/acc1 += A[ra..ra+1][cbeg..cend) . x
// STR: 0 default policy (__ldg), 1 streaming (evict-first), 2 keep (L2 evict-last hint `pol`)
template <int STR, bool XS, int UNROLL>
__device__ __forceinline__ void gemv_unit(const double2* __restrict__ a0, const double2* __restrict__ a1, int cbeg, int cend,
                                          int lane, const double* xs, double& acc0, double& acc1, unsigned long long pol = 0)
{
    auto ld = [&](const double2* q) { return STR == 2 ? gemv_ld_hint(q, pol) : (STR == 1 ? __ldcs(q) : __ldg(q)); };
    int c = cbeg + lane;
    for (; c + 32 * (UNROLL - 1) < cend; c += 32 * UNROLL) {
        double2 v0[UNROLL], v1[UNROLL];
#pragma unroll
        for (int i = 0; i < UNROLL; ++i) {
            v0[i] = ld(a0 + c + 32 * i);
            v1[i] = ld(a1 + c + 32 * i);
        }
#pragma unroll
        for (int i = 0; i < UNROLL; ++i) {
            double2 xv;
            if (XS) xv = reinterpret_cast<const double2*>(xs)[c + 32 * i];
            else xv = __ldcg(reinterpret_cast<const double2*>(xs) + c + 32 * i);
            acc0 = fma(v0[i].x, xv.x, acc0); acc0 = fma(v0[i].y, xv.y, acc0);
            acc1 = fma(v1[i].x, xv.x, acc1); acc1 = fma(v1[i].y, xv.y, acc1);
        }
    }
    for (; c < cend; c += 32) {
        const double2 v0 = ld(a0 + c), v1 = ld(a1 + c);
        double2 xv;
        if (XS) xv = reinterpret_cast<const double2*>(xs)[c];
        else xv = __ldcg(reinterpret_cast<const double2*>(xs) + c);
        acc0 = fma(v0.x, xv.x, acc0); acc0 = fma(v0.y, xv.y, acc0);
        acc1 = fma(v1.x, xv.x, acc1); acc1 = fma(v1.y, xv.y, acc1);
    }
}

// res_pairs (STREAM only): the first res_pairs row pairs of the CTA's block are read with the default cache policy and stay
// in the 126 MB L2 from one application to the next; the others are streamed (evict-first) so that they do not displace
// them.  For a matrix a little larger than L2 (n = 3500 ... 7000) this removes most of the HBM traffic of a GEMV.
template <bool STREAM, bool XS, int UNROLL = GEMV_UNROLL>
__device__ __forceinline__ void bie_cta_gemv(const double* __restrict__ A, long long lda, int n, int r0, int r1, int chunk,
                                             const double* xs, double* part, double* y_local, const Team& tm,
                                             int res_pairs = 0)
{
    const int lane = tm.tid & 31, warp = tm.warp, nwarp = tm.nwarp;
    const int rows = r1 - r0;
    const int rows2 = (rows + 1) & ~1;
    const int npair = rows2 >> 1;
    const int nch = (n + chunk - 1) / chunk;
    const int nunit = npair * nch;
    const int n2 = n >> 1;  // double2 columns (lda even: every row is 16-byte aligned)
    unsigned long long keep = 0;
    if (STREAM && res_pairs > 0) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(keep));
    for (int u = warp; u < nunit; u += nwarp) {
        // consecutive warps take consecutive chunks of the same row pair
        const int p = u / nch, ch = u - p * nch;
        const int ra = r0 + 2 * p;
        const bool two = (ra + 1 < r1);
        const double2* a0 = reinterpret_cast<const double2*>(A + (long long)ra * lda);
        const double2* a1 = reinterpret_cast<const double2*>(A + (long long)(two ? ra + 1 : ra) * lda);
        const int cbeg = ch * (chunk >> 1);
        const int cend = min(cbeg + (chunk >> 1), n2);
        double acc0 = 0.0, acc1 = 0.0;
        if (STREAM && p >= res_pairs) gemv_unit<1, XS, UNROLL>(a0, a1, cbeg, cend, lane, xs, acc0, acc1);
        else if (STREAM) gemv_unit<2, XS, UNROLL>(a0, a1, cbeg, cend, lane, xs, acc0, acc1, keep);
        else gemv_unit<0, XS, UNROLL>(a0, a1, cbeg, cend, lane, xs, acc0, acc1);
        if ((n & 1) && ch == nch - 1 && lane == 0) {  // odd n: the last column
            const double xl = XS ? xs[n - 1] : __ldcg(xs + n - 1);
            acc0 = fma(A[(long long)ra * lda + n - 1], xl, acc0);
            if (two) acc1 = fma(A[(long long)(ra + 1) * lda + n - 1], xl, acc1);
        }
        acc0 = bie_warp_sum(acc0);
        acc1 = bie_warp_sum(acc1);
        if (lane == 0) {
            part[ch * rows2 + 2 * p] = acc0;
            part[ch * rows2 + 2 * p + 1] = acc1;
        }
    }
    team_sync(tm);
    for (int r = tm.tid; r < rows; r += tm.nthr) {
        double s = 0.0;
        for (int ch = 0; ch < nch; ++ch) s += part[ch * rows2 + r];
        y_local[r] = s;
    }
    team_sync(tm);
}
