// bie_build.cu -- SURVEY 8(a) rows a2-a4: the dense collocation matrix of Eq. (3.16).
//
// Tiling.  A CTA of 128 threads owns a tile of T target rows x 256 source columns.  Each thread keeps the
// per-node factors of TWO adjacent source columns in registers and walks down the T target rows, whose
// factors (S, C, P, N) sit in shared memory and are read as warp-wide broadcasts.  A warp therefore writes,
// per target row, 32 x 16 B = 512 contiguous bytes of that row (128-bit coalesced stores, full 128 B lines).
//
// Per pair (fast path): 19 FP64-pipe instructions + 1 MUFU, no transcendental (bie_common.cuh).
// The walk over the target rows is split into segments of constant target component, so that the
// Re/Im selection of Eq. (3.10) and the -1/M_k of E_k become two
// per-segment register coefficients (u, v) and one fused constant em:
//     entry = (u * nr + v * ni) * r - em,      c = q * cot(w/2),  cot = (nr - i ni) r
//     Im c  ->  (u, v) = ( qi, -qr)      [k = 0, j = 0]  and  [k >= 1, j >= 1]
//     Re c  ->  (u, v) = ( qr,  qi)      [k = 0, j >= 1]
//    -Re c  ->  (u, v) = (-qr, -qi)      [k >= 1, j = 0]
// Pairs closer than |w|^2 < BIE_NEAR_TAU (which includes s == t) take the near path: Laurent series of
// cot from the coordinate differences, or the precomputed diagonal entry when s == t.
#include "bie_common.cuh"

#define BUILD_THREADS 128
#define BUILD_COLS 2
#define BUILD_TILE_W (BUILD_THREADS * BUILD_COLS)

struct SrcRegs {
    double S2, C2, P, N;  // 2 sin(x_s/2), 2 cos(x_s/2), e^{y_s/2}, e^{-y_s/2}
    double qr, qi;
    double u, v, em;  // per-segment coefficients
};

__device__ __forceinline__ double bie_pair_entry(const SrcRegs& s, const double2 sc, const double2 pn,
                                                 const NodeTable& nt, int sidx, int tidx)
{
    // 2 sin a = (2 S_s) C_t - (2 C_s) S_t ; 2 cos a = (2 C_s) C_t + (2 S_s) S_t
    const double sa = fma(s.S2, sc.y, -(s.C2 * sc.x));
    const double ca = fma(s.C2, sc.y, s.S2 * sc.x);
    const double ep = s.P * pn.y, en = s.N * pn.x;
    const double D = ep - en, G = ep + en;
    double nr = sa * ca, ni = D * G;
    const double den = fma(D, D, sa * sa);
    double r = bie_rcp(den);
    if (den < BIE_NEAR_TAU) {
        if (sidx == tidx) return nt.DIAG[tidx];
        double cr, ci;
        bie_cot_half_near(nt.X[sidx] - nt.X[tidx], nt.Y[sidx] - nt.Y[tidx], &cr, &ci);
        nr = cr; ni = -ci; r = 1.0;
    }
    return fma(fma(s.v, ni, s.u * nr), r, -s.em);
}

__global__ void __launch_bounds__(BUILD_THREADS)
bie_build_kernel(NodeTable nt, CompTable ct, double* __restrict__ A, long long lda, int T, int only0)
{
    extern __shared__ __align__(16) double2 sm[];  // [T] (S_t, C_t) then [T] (P_t, N_t)
    const int n = nt.n;
    const int c0 = blockIdx.x * BUILD_TILE_W;
    const int t0 = blockIdx.y * T;
    const int t1 = min(t0 + T, n);
    if (only0 && t0 >= ct.off[1] && c0 >= ct.off[1]) return;  // a4: solid-solid tiles stay
    double2* sSC = sm;
    double2* sPN = sm + T;
    for (int i = threadIdx.x; i < t1 - t0; i += BUILD_THREADS) {
        sSC[i] = make_double2(nt.S[t0 + i], nt.C[t0 + i]);
        sPN[i] = make_double2(nt.P[t0 + i], nt.N[t0 + i]);
    }
    const int s0 = c0 + BUILD_COLS * threadIdx.x;  // < npad by construction
    SrcRegs src[BUILD_COLS];
    int scomp[BUILD_COLS];
    double sem[BUILD_COLS];
#pragma unroll
    for (int c = 0; c < BUILD_COLS; ++c) {
        src[c].S2 = 2.0 * nt.S[s0 + c];
        src[c].C2 = 2.0 * nt.C[s0 + c];
        src[c].P = nt.P[s0 + c];
        src[c].N = nt.N[s0 + c];
        src[c].qr = nt.QR[s0 + c];
        src[c].qi = nt.QI[s0 + c];
        sem[c] = nt.EM[s0 + c];
        scomp[c] = nt.COMP[s0 + c];
    }
    __syncthreads();
    const bool full = (s0 + 1 < n);
    const bool part = (s0 < n);
    for (int k = 0; k < ct.ncomp; ++k) {
        const int a = max(t0, ct.off[k]), b = min(t1, ct.off[k + 1]);
        if (a >= b) continue;
#pragma unroll
        for (int c = 0; c < BUILD_COLS; ++c) {
            const bool src0 = (scomp[c] == 0), tgt0 = (k == 0);
            if (src0 == tgt0) { src[c].u = src[c].qi; src[c].v = -src[c].qr; }        // Im c
            else if (tgt0)    { src[c].u = src[c].qr; src[c].v = src[c].qi; }         // Re c   (G_0j)
            else              { src[c].u = -src[c].qr; src[c].v = -src[c].qi; }       // -Re c  (-G_k0)
            src[c].em = (scomp[c] == k) ? sem[c] : 0.0;
        }
        double* row = A + (long long)a * lda + s0;
#pragma unroll 2
        for (int t = a; t < b; ++t, row += lda) {
            const double2 sc = sSC[t - t0], pn = sPN[t - t0];
            const double e0 = bie_pair_entry(src[0], sc, pn, nt, s0, t);
            const double e1 = bie_pair_entry(src[1], sc, pn, nt, s0 + 1, t);
            if (full) *reinterpret_cast<double2*>(row) = make_double2(e0, e1);
            else if (part) row[0] = e0;
        }
    }
}

int bie_launch_build(bie_ctx* ctx, double* A, int64_t lda, int only_comp0, cudaStream_t st)
{
    if (!ctx || !A) return BIE_ERR_NULL;
    if (!ctx->have_geom) return BIE_ERR_GEOMETRY;
    const int n = ctx->n;
    if (lda < n || (lda & 1) || (((uintptr_t)A) & 15u)) return BIE_ERR_LAYOUT;
    const NodeTable nt = bie_node_table(ctx);
    const int gx = nt.npad / BUILD_TILE_W;
    // rows per CTA: 128 when that still gives every SM several CTAs, else smaller
    int T = 128;
    while (T > 8 && (long long)gx * ((n + T - 1) / T) < 4LL * ctx->sm_count) T >>= 1;
    dim3 grid(gx, (n + T - 1) / T);
    bie_build_kernel<<<grid, BUILD_THREADS, sizeof(double2) * 2 * T, st>>>(nt, ctx->comps, A, (long long)lda, T,
                                                                        only_comp0);
    BIE_CUDA(cudaGetLastError());
    return BIE_OK;
}
