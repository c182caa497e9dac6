// bie_nodes.cu -- SURVEY 8(a) row a1: per-node factors of the pair arithmetic (see bie_common.cuh).
//
// One thread per node.  The only transcendentals of the whole matrix build are evaluated here, O(n) of
// them: sincos(x) and exp(-(y - y_ref)), giving E = e^{i zeta} up to the common factor e^{-y_ref}
// (y_ref = Im zeta[0]; cot((zeta_s - zeta_t)/2) only sees ratios E_s/E_t).  Also the source weight
// q = zeta'/(2 M_j), the near threshold thr = tau_s |E|^2, and the complete diagonal entry from the
// limit K_jj(a,a) = Im{zeta''/(2 zeta')} with the -+1/2 of Eq. (3.10) and the
// -1/M_m of E_m.
#include "bie_common.cuh"
#include <cstdlib>
#include "bie_free.cuh"

struct PrepArgs {
    CompTable comps;
    int kinds[BIE_MAX_COMP];
};

__global__ void __launch_bounds__(256)
bie_prepare_nodes_kernel(PrepArgs pa, int n, int npad, int variant,
                         const double2* __restrict__ zeta, const double2* __restrict__ dzeta,
                         const double2* __restrict__ d2zeta, double2* __restrict__ buf, int* __restrict__ comp,
                         double2* __restrict__ T, double* __restrict__ taubar, double* __restrict__ kappa)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= npad) return;
    double2* E = buf;
    double2* MT = buf + (size_t)npad;
    double2* Q = buf + 2 * (size_t)npad;
    double2* XY = buf + 3 * (size_t)npad;
    double2* DG = buf + 4 * (size_t)npad;
    if (i >= n) {  // padding: zero weight, never near (thr = 0), never stored to A
        E[i] = make_double2(0.0, 0.0); MT[i] = make_double2(0.0, 0.0); Q[i] = make_double2(0.0, 0.0);
        XY[i] = make_double2(0.0, 1.0e3); DG[i] = make_double2(0.0, 0.0); comp[i] = -1;
        // padding sources of the matrix-free tables: zero weight for every vector
        for (int a = 0; a < 4; ++a) T[(size_t)a * npad + i] = make_double2(0.0, 0.0);
        return;
    }
    int k = 0;
    while (k + 1 < pa.comps.ncomp && i >= pa.comps.off[k + 1]) ++k;
    const double M = (double)(pa.comps.off[k + 1] - pa.comps.off[k]);
    const double2 z = zeta[i], dz = dzeta[i], d2 = d2zeta[i];
    const double yref = zeta[0].y;
    double s, c;
    sincos(z.x, &s, &c);
    const double m = exp(-(z.y - yref));
    E[i] = make_double2(m * c, m * s);
    const double qr = dz.x / (2.0 * M), qi = dz.y / (2.0 * M);
    Q[i] = make_double2(qr, qi);
    double tau = BIE_NEAR_C * sqrt(qr * qr + qi * qi);
    tau = fmin(fmax(tau, BIE_NEAR_TAU_MIN), BIE_NEAR_TAU_MAX);
    MT[i] = make_double2(m * m, tau * m * m);
    // taubar = max_s tau_s (positive doubles order like their bit patterns)
    atomicMax(reinterpret_cast<unsigned long long*>(taubar), (unsigned long long)__double_as_longlong(tau));
    XY[i] = z;
    // Im{ zeta'' / (2 zeta' M) }
    const double den = dz.x * dz.x + dz.y * dz.y;
    double d = (d2.y * dz.x - d2.x * dz.y) / den / (2.0 * M);
    const double em = (variant == BIE_VARIANT_A && pa.kinds[k] == BIE_KIND_OBSTACLE) ? 1.0 / M : 0.0;
    // -1/2 I + K_00, 1/2 I + K_kk (Eq. 3.10); the vortex-sheet system has 1/2 I + K+_00, -1/2 I + K+_kk (Eqs. 4.14, 4.5)
    if (variant == BIE_VARIANT_NORMAL_INTERNAL) {
        // normal-velocity operator (Section 3.4): diagonal -G_00(a,a)/M_0 = -Re{zeta''/(2 zeta')}/M_0,
        // and the real-cot table kappa_d, d = m - l mod M_0, that carries the regulariser of G_00 and
        // -1/2 of the discrete Hilbert transform (symbol -i sgn k) together:
        //   M_0 even: (-1)^d cot(pi d/M_0)/(2 M_0)      M_0 odd: (-1)^d / (2 M_0 sin(pi d/M_0))      kappa_0 = 0
        d = -(d2.x * dz.x + d2.y * dz.y) / den / (2.0 * M);
        if (k == 0) {
            double kv = 0.0;
            if (i > 0) {
                const int M0 = pa.comps.off[1];
                const double sgn = (i & 1) ? -1.0 : 1.0;
                const double sp = sinpi((double)i / M), cp = cospi((double)i / M);
                kv = (M0 & 1) ? sgn / (2.0 * M * sp) : sgn * cp / (2.0 * M * sp);
            }
            kappa[i] = kv;
        }
    } else if (variant == BIE_VARIANT_VORTEX) d += (k == 0) ? 0.5 : -0.5;
    else d += (k == 0) ? -0.5 : 0.5;
    d -= em;
    DG[i] = make_double2(d, em);
    comp[i] = k;
}

NodeTable bie_node_table(const bie_ctx* ctx)
{
    NodeTable t;
    const size_t np = (size_t)bie_npad(ctx->n);
    const double2* b = reinterpret_cast<const double2*>(ctx->node_buf);
    t.E = b;
    t.MT = b + np;
    t.Q = b + 2 * np;
    t.XY = b + 3 * np;
    t.DG = b + 4 * np;
    t.COMP = ctx->comp_buf;
    t.n = ctx->n;
    t.npad = (int)np;
    return t;
}

int bie_prepare_nodes(bie_ctx* ctx, int ncomp, const int32_t* counts, const int32_t* kinds,
                      const double* zeta, const double* dzeta, const double* d2zeta, int variant,
                      cudaStream_t st)
{
    if (!ctx || !counts || !kinds || !zeta || !dzeta || !d2zeta) return BIE_ERR_NULL;
    if (ncomp < 1 || ncomp > BIE_MAX_COMP) return BIE_ERR_GEOMETRY;
    if (variant != BIE_VARIANT_A && variant != BIE_VARIANT_B && variant != BIE_VARIANT_VORTEX &&
        variant != BIE_VARIANT_NORMAL_INTERNAL) return BIE_ERR_ARG;
    long long n = 0;
    int nbottom = 0;
    for (int c = 0; c < ncomp; ++c) {
        if (counts[c] < 1) return BIE_ERR_GEOMETRY;
        if (kinds[c] < 0 || kinds[c] > 2) return BIE_ERR_GEOMETRY;
        if ((kinds[c] == BIE_KIND_SURFACE) != (c == 0)) return BIE_ERR_GEOMETRY;
        if (kinds[c] == BIE_KIND_BOTTOM) ++nbottom;
        n += counts[c];
    }
    if (nbottom > 1 || n > (1 << 30)) return BIE_ERR_GEOMETRY;
    if ((((uintptr_t)zeta) | ((uintptr_t)dzeta) | ((uintptr_t)d2zeta)) & 15u) return BIE_ERR_LAYOUT;
    const int npad = bie_npad((int)n);
    ctx->geom_gen += 1;          // whatever was cached for the previous geometry (near matrix, symmetric work list) is stale
    ctx->near_valid = 0;
    if (npad > ctx->cap) {
        // grow the ctx's node storage (O(n) bytes).  The ctx holds NO geometry until every allocation and the
        // preparation launch below have succeeded.
        ctx->have_geom = 0; ctx->n = 0;
        if (ctx->node_buf) cudaFree(ctx->node_buf);
        if (ctx->comp_buf) cudaFree(ctx->comp_buf);
        if (ctx->free_buf) cudaFree(ctx->free_buf);
        if (ctx->near_ptr) cudaFree(ctx->near_ptr);
        if (ctx->kappa) cudaFree(ctx->kappa);
        ctx->kappa = nullptr;
        ctx->node_buf = nullptr; ctx->comp_buf = nullptr; ctx->free_buf = nullptr; ctx->cap = 0;
        ctx->near_ptr = nullptr;
        cudaError_t e = cudaMalloc((void**)&ctx->node_buf, sizeof(double) * BIE_NODE_ARRAYS * (size_t)npad);
        if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->comp_buf, sizeof(int) * (size_t)npad);
        if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->free_buf, sizeof(double) * bie_free_buf_doubles(npad));
        if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->near_ptr, sizeof(int) * (8 * (size_t)npad + 4));
        if (e == cudaSuccess) e = cudaMalloc((void**)&ctx->kappa, sizeof(double) * (size_t)npad);
        if (e != cudaSuccess) {
            cudaGetLastError();   // clear the sticky-free allocation error; the ctx stays without a geometry
            return bie_cuda_err(e);
        }
        ctx->cap = npad;
    }
    PrepArgs pa;
    pa.comps.ncomp = ncomp;
    pa.comps.off[0] = 0;
    for (int c = 0; c < BIE_MAX_COMP; ++c) {
        pa.kinds[c] = c < ncomp ? kinds[c] : 0;
        pa.comps.off[c + 1] = c < ncomp ? pa.comps.off[c] + counts[c] : (int)n;
    }
    ctx->have_geom = 0;
    BIE_CUDA(cudaMemsetAsync(ctx->taubar, 0, sizeof(double), st));
    bie_prepare_nodes_kernel<<<(npad + 255) / 256, 256, 0, st>>>(
        pa, (int)n, npad, variant, (const double2*)zeta, (const double2*)dzeta, (const double2*)d2zeta,
        (double2*)ctx->node_buf, ctx->comp_buf, (double2*)ctx->free_buf, ctx->taubar, ctx->kappa);
    BIE_CUDA(cudaGetLastError());
    ctx->n = (int)n;
    ctx->ncomp = ncomp;
    ctx->variant = variant;
    for (int c = 0; c < ncomp; ++c) { ctx->counts[c] = counts[c]; ctx->kinds[c] = kinds[c]; }
    ctx->comps = pa.comps;
    ctx->have_geom = 1;
    return BIE_OK;
}

// ---- matrix-free operator: storage and work split (bie_free.cuh) ------------------------------------------
size_t bie_free_buf_doubles(int cap)
{
    // tables [4][cap] double2, then partial sums for (row blocks + CTAs) parts of FREE_ROWS rows, then the per-CTA
    // partials of the constant terms [4][FREE_SB_LD]
    return 8 * (size_t)cap + ((size_t)cap / FREE_ROWS + 2 + 256) * FREE_ROWS + 2 * 4 * FREE_SB_LD;
}

// work list of the symmetric split (bie_free_sym.cuh), built on the device by one thread (NB <= a few hundred):
// blocks in the order 0, NB-1, 1, NB-2, ... (long and short source lists alternate); cum[k] = sources before position k
__global__ void bie_sym_tables_kernel(int NB, int NB0, int M0, int n, int npad, int s_off, int first, long long* cum,
                                      int* perm, int* pos)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    long long c = 0;
    cum[0] = 0;
    for (int k = 0; k < NB; ++k) {
        const int b = (k & 1) ? NB - 1 - (k >> 1) : (k >> 1);
        perm[k] = b;
        pos[b] = k;
        const int row0 = b < NB0 ? b * FREE_ROWS : M0 + (b - NB0) * FREE_ROWS;
        const int src0 = b < first ? s_off : row0;
        c += SYM_PART_PAD + (npad - src0);     // + the virtual sources that stand for the fixed cost of a part
        cum[k + 1] = c;
    }
    (void)n;
}

int bie_free_plan(bie_ctx* ctx, int grid, int s_off, FreePlan* fp, cudaStream_t st)
{
    if (!ctx->have_geom || grid < 1 || grid > 256) return BIE_ERR_GEOMETRY;
    if (ctx->variant == BIE_VARIANT_NORMAL_INTERNAL) return BIE_ERR_GEOMETRY;   // node tables of another operator
    if (s_off < 0 || (s_off & 1) || s_off > ctx->n) return BIE_ERR_ARG;
    const int n = ctx->n, npad = bie_npad(n);
    fp->M0 = ctx->counts[0];
    fp->NB0 = (fp->M0 + FREE_ROWS - 1) / FREE_ROWS;
    fp->NB = fp->NB0 + (n - fp->M0 + FREE_ROWS - 1) / FREE_ROWS;
    fp->vortex = (ctx->variant == BIE_VARIANT_VORTEX) ? 1 : 0;
    fp->s_off = s_off;
    // hybrid operator: s_off must be a row-block boundary (row blocks are cut per class: 128 b, then M_0 + 128 b)
    const bool boundary = s_off == 0 || (s_off <= fp->M0 ? (s_off % FREE_ROWS == 0 || s_off == fp->M0)
                                                          : ((s_off - fp->M0) % FREE_ROWS == 0));
    if (!boundary) return BIE_ERR_ARG;
    auto row0_of = [&](int b) { return b < fp->NB0 ? b * FREE_ROWS : fp->M0 + (b - fp->NB0) * FREE_ROWS; };
    auto rows_of = [&](int b) { const int r0 = row0_of(b), end = b < fp->NB0 ? fp->M0 : n; return end - r0 < FREE_ROWS ? end - r0 : FREE_ROWS; };
    int first = 0;   // row blocks entirely below s_off: they only take the sources from s_off on (the stored block has the others)
    while (first < fp->NB && row0_of(first) + rows_of(first) <= s_off) ++first;
    fp->nb_below = first;
    fp->UBb = (npad - s_off) / 2;
    fp->UBf = npad / 2;
    fp->U = (long long)first * fp->UBb + (long long)(fp->NB - first) * fp->UBf;
    // symmetric work split (bie_free_sym.cuh): Eq. (3.16) variants, and while the reverse partials [NB][npad] stay small
    fp->sym = 0; fp->PC = nullptr; fp->sym_cum = nullptr; fp->sym_perm = nullptr; fp->sym_pos = nullptr;
    if (bie_uses_sym(ctx)) {
        const int NB = fp->NB;
        const size_t need = (size_t)NB * (size_t)npad;
        if (need > ctx->pc_cap) {
            if (ctx->pc_buf) cudaFree(ctx->pc_buf);
            ctx->pc_buf = nullptr; ctx->pc_cap = 0;
            if (cudaMalloc((void**)&ctx->pc_buf, sizeof(double) * need) != cudaSuccess) {
                cudaGetLastError();
                return BIE_ERR_CUDA_BASE - (int)cudaErrorMemoryAllocation;
            }
            ctx->pc_cap = need;
        }
        // the tables are cached per (geometry, s_off): cum [NB + 1] long long, perm [NB], pos [NB]; sized for the largest
        // NB the node capacity allows
        const size_t nbmax = (size_t)ctx->cap / FREE_ROWS + 4;
        const size_t tab_bytes = sizeof(long long) * (nbmax + 1) + 2 * sizeof(int) * nbmax;
        if (tab_bytes > ctx->sym_tab_bytes) {
            if (ctx->sym_tab) cudaFree(ctx->sym_tab);
            ctx->sym_tab = nullptr; ctx->sym_tab_bytes = 0; ctx->sym_key[0] = -1;
            if (cudaMalloc((void**)&ctx->sym_tab, tab_bytes) != cudaSuccess) {
                cudaGetLastError();
                return BIE_ERR_CUDA_BASE - (int)cudaErrorMemoryAllocation;
            }
            ctx->sym_tab_bytes = tab_bytes;
        }
        long long* cum = reinterpret_cast<long long*>(ctx->sym_tab);
        int* perm = reinterpret_cast<int*>(ctx->sym_tab + sizeof(long long) * (nbmax + 1));
        int* pos = perm + nbmax;
        if (ctx->sym_key[0] != ctx->geom_gen || ctx->sym_key[1] != s_off) {
            long long U = 0;
            for (int b = 0; b < NB; ++b) U += SYM_PART_PAD + npad - (b < first ? s_off : row0_of(b));
            bie_sym_tables_kernel<<<1, 32, 0, st>>>(NB, fp->NB0, fp->M0, n, npad, s_off, first, cum, perm, pos);
            BIE_CUDA(cudaGetLastError());
            ctx->sym_key[0] = ctx->geom_gen; ctx->sym_key[1] = s_off;
            ctx->sym_U = U;
        }
        fp->sym_cum = cum; fp->sym_perm = perm; fp->sym_pos = pos;
        fp->sym = 1; fp->PC = ctx->pc_buf; fp->U = ctx->sym_U;
    }
    fp->stage_buf = free_stage_buf_doubles(fp->vortex != 0, fp->sym != 0);
    fp->Geff = (long long)grid < fp->U ? grid : (int)fp->U;
    if (fp->Geff < 1) fp->Geff = 1;
    fp->T = reinterpret_cast<double2*>(ctx->free_buf);
    fp->PB = ctx->free_buf + 8 * (size_t)npad;
    fp->SB = ctx->free_buf + 8 * (size_t)ctx->cap + ((size_t)ctx->cap / FREE_ROWS + 2 + 256) * FREE_ROWS;
    fp->taubar = ctx->taubar;
    fp->near_ptr = ctx->near_ptr; fp->near_col = ctx->near_col; fp->near_val = ctx->near_val;
    return BIE_OK;
}
