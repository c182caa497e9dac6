// bie_eval.cu -- SURVEY 8(f) NEXT-3, Section 5.1 / Appendix F: values inside the fluid,
// up to the boundary, of functions analytic in the fluid from their boundary values (Helsing & Ojala, periodic form):
//     f(z) ~ sum_s lambda~_s(z) f_s / sum_s lambda~_s(z),    lambda~_s(z) = (sigma_k/M_k) 1/2 cot((zeta_s - z)/2) zeta'_s   (F.4)/(5.5)
// sigma_0 = -1 on Gamma_0 (fluid on its right; reading R18), +1 on the solids.  "If z coincides with
// zeta_k(alpha_m), we set f(z) = f(zeta_k(alpha_m))".
//
// Second workload of the same pair arithmetic (bie_common.cuh), in its difference form: with d = E_s - E_z = dr + i di,
//     q_s cot((zeta_s - z)/2) = (A_s dr + B_s di)/den - i q_s,     A_s = 2 i q_s E_s,  B_s = 2 q_s E_s = -i A_s,
// so with u = dr/den, v = di/den every complex sum (the denominator and the nf numerators, whose source constant is A_s f_s)
// costs 4 FMAs per pair:  Re += Ar u + Ai v,  Im += Ai u - Ar v;  the constants -i sum_s q_s (f_s) are added per source tile by
// one thread.  Per pair: 2 sub, 2 den, 3 reciprocal, 2 for (u, v), 4 per sum = 9 + 4 (1 + nf) FP64 instructions (12 + 4 (1 + nf)
// with the (X, Y) form of round 1).  Three or four evaluation points per thread share every shared-memory load (eval_np);
// the sources are staged tile by tile in shared memory with E_s, the near threshold and
// A_s, A_s f_s.  Pairs closer than the near threshold are recomputed from the coordinate differences
// with the Laurent series (exact to rounding at any distance, which is the whole point of (F.4)); an exact coincidence
// is recorded and resolved in the second kernel, which also adds the partial sums of the source segments (few points:
// the sources are split over blockIdx.y so that the GPU is filled) and divides.
#include "bie_common.cuh"

#define EVAL_THREADS 128
#define EVAL_TILE 256
#define EVAL_MAX_NF 4

struct EvalComps {
    int ncomp;
    int off[BIE_MAX_COMP + 1];
    int surface[BIE_MAX_COMP];   // 1: sigma = -1
};

// evaluation points per thread (they share every shared-memory load): measured at 65 536 points x 16 384 sources, as a share of
// the probed FP64 rate, (points, resident CTAs) = (2, 4) / (4, 3) / (3, 3): nf = 1 0.68 / 0.71 / 0.68, nf = 2 0.67 / 0.72 / 0.67,
// nf = 4 0.70 / 0.69 / 0.71
static inline int eval_np(int nf) { return nf <= 2 ? 4 : 3; }
#ifndef EVAL_UNROLL
#define EVAL_UNROLL 2  // sources per unrolled step of the fast pass
#endif
constexpr int kEvalUnroll = EVAL_UNROLL;
#ifndef EVAL_RESIDENT
#define EVAL_RESIDENT 3   // CTAs per SM the register allocation must allow; eval_nseg() fills whole waves of them
#endif

template <int NF, int EVAL_NP>
__global__ void __launch_bounds__(EVAL_THREADS, EVAL_RESIDENT)
bie_cauchy_eval_kernel(EvalComps ec, int n, const double2* __restrict__ zeta, const double2* __restrict__ dzeta,
                       const double2* __restrict__ f, int npts, const double2* __restrict__ zpts, int nseg,
                       double2* __restrict__ part /* [nseg][1+NF][npts] */, int* __restrict__ hit /* [npts] */)
{
    __shared__ double2 sE[EVAL_TILE], sA[EVAL_TILE], sQ[EVAL_TILE], sXY[EVAL_TILE];
    __shared__ double2 sG[NF][EVAL_TILE];
    __shared__ int sTH[EVAL_TILE];
    __shared__ double2 sred[EVAL_THREADS / 32][1 + NF];
    const int seg = blockIdx.y;
    const int per = (((n + nseg - 1) / nseg) + 1) & ~1;
    const int s_lo = seg * per, s_hi = min(s_lo + per, n);
    const double yref = zeta[0].y;
    // this thread's points: p0 + k EVAL_THREADS (consecutive threads, consecutive points)
    const int p0 = blockIdx.x * (EVAL_THREADS * EVAL_NP) + threadIdx.x;
    double2 z[EVAL_NP];
    double ter[EVAL_NP], tei[EVAL_NP];
    double Dr[EVAL_NP], Di[EVAL_NP], Nr[EVAL_NP][NF], Ni[EVAL_NP][NF];
    int myhit[EVAL_NP];
#pragma unroll
    for (int k = 0; k < EVAL_NP; ++k) {
        z[k] = zpts[min(p0 + k * EVAL_THREADS, npts - 1)];
        double s, c;
        sincos(z[k].x, &s, &c);
        const double m = exp(-(z[k].y - yref));
        ter[k] = m * c; tei[k] = m * s;
        Dr[k] = 0.0; Di[k] = 0.0; myhit[k] = -1;
#pragma unroll
        for (int q = 0; q < NF; ++q) { Nr[k][q] = 0.0; Ni[k][q] = 0.0; }
    }
    // sum_s q_s and sum_s q_s f_s over the segment (the constant -i q_s of the difference form), this thread's share
    double2 cs[1 + NF];
#pragma unroll
    for (int c = 0; c <= NF; ++c) cs[c] = make_double2(0.0, 0.0);
    for (int s0 = s_lo; s0 < s_hi; s0 += EVAL_TILE) {
        __syncthreads();
        for (int i = threadIdx.x; i < EVAL_TILE; i += EVAL_THREADS) {
            const int s = s0 + i;
            if (s < s_hi) {
                int k = 0;
                while (k + 1 < ec.ncomp && s >= ec.off[k + 1]) ++k;
                const double M = (double)(ec.off[k + 1] - ec.off[k]);
                const double wgt = (ec.surface[k] ? -0.5 : 0.5) / M;
                const double2 zs = zeta[s], dz = dzeta[s];
                double sn, cn;
                sincos(zs.x, &sn, &cn);
                const double m = exp(-(zs.y - yref));
                const double2 q = make_double2(wgt * dz.x, wgt * dz.y);
                double tau = BIE_NEAR_C * sqrt(q.x * q.x + q.y * q.y);
                tau = fmin(fmax(tau, BIE_NEAR_TAU_MIN), BIE_NEAR_TAU_MAX);
                const double er = m * cn, ei = m * sn;
                // A_s = 2 i q_s E_s
                const double qer = q.x * er - q.y * ei, qei = q.x * ei + q.y * er;     // q E
                const double2 A = make_double2(-2.0 * qei, 2.0 * qer);
                sE[i] = make_double2(er, ei);
                sTH[i] = __double2hiint(tau * m * m);
                sA[i] = A;
                sQ[i] = q;
                sXY[i] = zs;
                cs[0].x += q.x; cs[0].y += q.y;
#pragma unroll
                for (int c = 0; c < NF; ++c) {
                    const double2 fv = f[(size_t)c * n + s];
                    sG[c][i] = make_double2(A.x * fv.x - A.y * fv.y, A.x * fv.y + A.y * fv.x);   // A_s f_s
                    cs[1 + c].x += q.x * fv.x - q.y * fv.y; cs[1 + c].y += q.x * fv.y + q.y * fv.x;
                }
            } else {   // beyond the segment: zero weight, never near
                sE[i] = make_double2(0.0, 0.0); sA[i] = make_double2(0.0, 0.0); sQ[i] = make_double2(0.0, 0.0);
                sXY[i] = make_double2(0.0, 1.0e3); sTH[i] = 0;
#pragma unroll
                for (int c = 0; c < NF; ++c) sG[c][i] = make_double2(0.0, 0.0);
            }
        }
        __syncthreads();
        // fast pass, branch-free: a near pair (rare) gets a ZERO reciprocal -- one select on the high word of the hardware
        // approximation, which the refinement of bie_rcp3 carries through (e = 1, r0 (1 + e + e^2) = 0) -- and raises a flag
        const int jn = min(EVAL_TILE, s_hi - s0);
        int flag[EVAL_NP];
#pragma unroll
        for (int k = 0; k < EVAL_NP; ++k) flag[k] = 0;
#pragma unroll kEvalUnroll
        for (int j = 0; j < jn; ++j) {
            const double2 e = sE[j], A = sA[j];
            const int th = sTH[j];
#pragma unroll
            for (int k = 0; k < EVAL_NP; ++k) {
                const double dr = e.x - ter[k], di = e.y - tei[k];
                const double den = fma(dr, dr, di * di);
                const bool near = __double2hiint(den) < th;
                flag[k] |= near ? 1 : 0;
                double r0;
                asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r0) : "d"(den));
                r0 = __hiloint2double(near ? 0 : __double2hiint(r0), 0);   // the approximation has a zero low word
                const double er_ = fma(-den, r0, 1.0);
                const double r = fma(r0, fma(er_, er_, er_), r0);
                const double u = dr * r, v = di * r;
                Dr[k] = fma(A.x, u, Dr[k]); Dr[k] = fma(A.y, v, Dr[k]);
                Di[k] = fma(A.y, u, Di[k]); Di[k] = fma(-A.x, v, Di[k]);
#pragma unroll
                for (int c = 0; c < NF; ++c) {
                    const double2 g = sG[c][j];
                    Nr[k][c] = fma(g.x, u, Nr[k][c]); Nr[k][c] = fma(g.y, v, Nr[k][c]);
                    Ni[k][c] = fma(g.y, u, Ni[k][c]); Ni[k][c] = fma(-g.x, v, Ni[k][c]);
                }
            }
        }
        // near pairs of this tile (threads that saw one revisit the tile): from the coordinate differences
#pragma unroll
        for (int k = 0; k < EVAL_NP; ++k) {
            if (!flag[k]) continue;
            for (int j = 0; j < jn; ++j) {
                const double2 e = sE[j];
                const double dr = e.x - ter[k], di = e.y - tei[k];
                const double den = fma(dr, dr, di * di);          // the same bits as in the fast pass
                if (__double2hiint(den) >= sTH[j]) continue;
                const double2 zs = sXY[j], q = sQ[j];
                const double x = zs.x - z[k].x, y = zs.y - z[k].y;
                // exact coincidence (modulo the period): cot has a pole, (F.4) degenerates to f_s
                const double xr = x - 6.283185307179586232 * rint(x * 0.15915494309189534561);
                if (xr == 0.0 && y == 0.0) { myhit[k] = s0 + j; continue; }
                double cr, ci;
                bie_cot_half_near(x, y, &cr, &ci);
                ci += 1.0;                             // + i q_s: the constant below is subtracted for EVERY source
                const double wr = q.x * cr - q.y * ci, wi = q.x * ci + q.y * cr;
                Dr[k] += wr; Di[k] += wi;
#pragma unroll
                for (int c = 0; c < NF; ++c) {
                    const double2 fv = f[(size_t)c * n + s0 + j];
                    Nr[k][c] += wr * fv.x - wi * fv.y; Ni[k][c] += wr * fv.y + wi * fv.x;
                }
            }
        }
    }
    // the constants: fixed-order sum over the CTA (lanes by shuffle, warps in order), then -i sum
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int c = 0; c <= NF; ++c) { cs[c].x = bie_warp_sum(cs[c].x); cs[c].y = bie_warp_sum(cs[c].y); }
    __syncthreads();
    if (lane == 0) {
#pragma unroll
        for (int c = 0; c <= NF; ++c) sred[warp][c] = cs[c];
    }
    __syncthreads();
#pragma unroll
    for (int c = 0; c <= NF; ++c) {
        double sx = 0.0, sy = 0.0;
        for (int w = 0; w < EVAL_THREADS / 32; ++w) { sx += sred[w][c].x; sy += sred[w][c].y; }
        cs[c] = make_double2(sx, sy);
    }
#pragma unroll
    for (int k = 0; k < EVAL_NP; ++k) {
        const int p = p0 + k * EVAL_THREADS;
        if (p < npts) {
            double2* o = part + (size_t)seg * (1 + NF) * npts;
            o[p] = make_double2(Dr[k] + cs[0].y, Di[k] - cs[0].x);        // - i (sx + i sy) = sy - i sx
#pragma unroll
            for (int c = 0; c < NF; ++c) o[(size_t)(1 + c) * npts + p] = make_double2(Nr[k][c] + cs[1 + c].y, Ni[k][c] - cs[1 + c].x);
            if (myhit[k] >= 0) atomicMax(hit + p, myhit[k]);
        }
    }
}

// out[c][p] = N_c / D (fixed-order sum over the source segments), or the boundary value at a coincident node
__global__ void __launch_bounds__(256)
bie_cauchy_finish_kernel(int nf, int n, int npts, int nseg, const double2* __restrict__ part, const int* __restrict__ hit,
                         const double2* __restrict__ f, double2* __restrict__ out)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npts) return;
    const int h = hit[p];
    double Dr = 0.0, Di = 0.0;
    for (int s = 0; s < nseg; ++s) {
        const double2 d = part[(size_t)s * (1 + nf) * npts + p];
        Dr += d.x; Di += d.y;
    }
    const double inv = 1.0 / (Dr * Dr + Di * Di);
    for (int c = 0; c < nf; ++c) {
        if (h >= 0) { out[(size_t)c * npts + p] = f[(size_t)c * n + h]; continue; }
        double Nr = 0.0, Ni = 0.0;
        for (int s = 0; s < nseg; ++s) {
            const double2 v = part[((size_t)s * (1 + nf) + 1 + c) * npts + p];
            Nr += v.x; Ni += v.y;
        }
        out[(size_t)c * npts + p] = make_double2((Nr * Dr + Ni * Di) * inv, (Ni * Dr - Nr * Di) * inv);
    }
}

// Source segments (blockIdx.y).  All CTAs take equally long (points per CTA x sources per segment), so the grid of
// gx x nseg CTAs should fill whole waves of sm_count x EVAL_RESIDENT resident CTAs: with the former rule (just enough CTAs
// for four per SM) 65 536 points gave 768 CTAs = 1.3 waves.  Smallest nseg that gives at least one wave and wastes < 3 %
// of the last one, else the best of 1 .. 64.
static int eval_nseg(int nf, int npts, int sm_count)
{
    const int gx = (npts + EVAL_THREADS * eval_np(nf) - 1) / (EVAL_THREADS * eval_np(nf));
    const long long wave = (long long)sm_count * EVAL_RESIDENT;
    int best = 1;
    double best_eff = 0.0;
    for (int s = 1; s <= 64; ++s) {
        const long long units = (long long)gx * s;
        const double eff = (double)units / (double)(((units + wave - 1) / wave) * wave);
        if (units >= wave && eff >= 0.97) return s;
        if (eff > best_eff + 1e-9) { best_eff = eff; best = s; }
    }
    return best;
}

size_t bie_cauchy_eval_ws_bytes(int nf, int npts, int sm_count)
{
    if (nf < 1 || nf > EVAL_MAX_NF || npts < 1) return 0;
    const int nseg = eval_nseg(nf, npts, sm_count);
    return sizeof(double2) * (size_t)nseg * (1 + nf) * npts + sizeof(int) * (size_t)npts + 256;
}

int bie_launch_cauchy_eval(bie_ctx* ctx, int ncomp, const int32_t* counts, const int32_t* kinds, const double* zeta,
                           const double* dzeta, int nf, const double* fvals, int npts, const double* zpts, double* out,
                           void* ws, size_t ws_bytes, cudaStream_t st)
{
    if (nf < 1 || nf > EVAL_MAX_NF || npts < 1) return BIE_ERR_ARG;
    if (!ctx || !counts || !kinds || !zeta || !dzeta || !fvals || !zpts || !out || !ws) return BIE_ERR_NULL;
    if (ncomp < 1 || ncomp > BIE_MAX_COMP) return BIE_ERR_GEOMETRY;
    EvalComps ec;
    ec.ncomp = ncomp; ec.off[0] = 0;
    long long n = 0;
    for (int c = 0; c < ncomp; ++c) {
        if (counts[c] < 1 || kinds[c] < 0 || kinds[c] > 2 || (kinds[c] == BIE_KIND_SURFACE) != (c == 0)) return BIE_ERR_GEOMETRY;
        n += counts[c];
        ec.off[c + 1] = (int)n; ec.surface[c] = (kinds[c] == BIE_KIND_SURFACE);
    }
    if (n > (1 << 30)) return BIE_ERR_GEOMETRY;
    if ((((uintptr_t)zeta) | ((uintptr_t)dzeta) | ((uintptr_t)fvals) | ((uintptr_t)zpts) | ((uintptr_t)out)) & 15u) return BIE_ERR_LAYOUT;
    if (bie_cauchy_eval_ws_bytes(nf, npts, ctx->sm_count) > ws_bytes) return BIE_ERR_WORKSPACE;
    const int gx = (npts + EVAL_THREADS * eval_np(nf) - 1) / (EVAL_THREADS * eval_np(nf));
    int nseg = eval_nseg(nf, npts, ctx->sm_count);
    if (nseg > (int)((n + 1) / 2)) nseg = (int)((n + 1) / 2);
    double2* part = (double2*)(((uintptr_t)ws + 255) & ~(uintptr_t)255);
    int* hit = (int*)(part + (size_t)nseg * (1 + nf) * npts);
    BIE_CUDA(cudaMemsetAsync(hit, 0xFF, sizeof(int) * (size_t)npts, st));
    dim3 grid(gx, nseg);
    const double2 *z2 = (const double2*)zeta, *d2 = (const double2*)dzeta, *f2 = (const double2*)fvals, *p2 = (const double2*)zpts;
    switch (nf) {
        case 1: bie_cauchy_eval_kernel<1, 4><<<grid, EVAL_THREADS, 0, st>>>(ec, (int)n, z2, d2, f2, npts, p2, nseg, part, hit); break;
        case 2: bie_cauchy_eval_kernel<2, 4><<<grid, EVAL_THREADS, 0, st>>>(ec, (int)n, z2, d2, f2, npts, p2, nseg, part, hit); break;
        case 3: bie_cauchy_eval_kernel<3, 3><<<grid, EVAL_THREADS, 0, st>>>(ec, (int)n, z2, d2, f2, npts, p2, nseg, part, hit); break;
        default: bie_cauchy_eval_kernel<4, 3><<<grid, EVAL_THREADS, 0, st>>>(ec, (int)n, z2, d2, f2, npts, p2, nseg, part, hit); break;
    }
    bie_cauchy_finish_kernel<<<(npts + 255) / 256, 256, 0, st>>>(nf, (int)n, npts, nseg, part, hit, f2, (double2*)out);
    BIE_CUDA(cudaGetLastError());
    return BIE_OK;
}
