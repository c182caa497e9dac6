// bie_cyl.cu -- SURVEY 8(f) NEXT-4, Appendix B: the variant in which the stream function is
// prescribed on the solid boundaries and the circulation parameters a_m = <1_m, omega> are unknowns.  Eq. (B.2)
// (PAPER.md:L1003):   A omega = B omega + sum_{m>=2} c_m <1_m, omega>,
//     c_m[t] = phi_cyl(zeta_t - z_m) for t on Gamma_0,  psi_cyl(zeta_t - z_m) for t on a solid,
//     Phi_cyl(z) = -i log(1 - e^{iz}) = phi_cyl + i psi_cyl  (Eq. (3.2)),
// and <1_m, omega> = (1/M_m) sum_l omega_m[l] on the trapezoidal rule: every column of obstacle m gets
// c_m[t]/M_m added in every row t.  The kernel ADDS this rank-(N-1) correction in place to a matrix that holds B
// (bie_build with BIE_VARIANT_B).  One warp per row and obstacle: the lanes sweep the obstacle's columns of that row
// (read-modify-write, coalesced); the transcendentals (one exp, sincos, and atan2 or log per row and obstacle) are
// O(n N) in total.  HBM-bound: 16 B per corrected entry.
#include <math.h>
#include "bie_common.cuh"

struct CylArgs {
    int nobs;
    int off[BIE_MAX_COMP];    // first column of obstacle o
    int cnt[BIE_MAX_COMP];    // M_m
    double zr[BIE_MAX_COMP], zi[BIE_MAX_COMP];
};

__global__ void __launch_bounds__(256)
bie_add_cyl_columns_kernel(CylArgs ca, int n, int M0, const double2* __restrict__ zeta, double* __restrict__ A, long long lda)
{
    const int lane = threadIdx.x & 31;
    const int t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);   // row
    const int o = blockIdx.y;                                             // obstacle
    if (t >= n) return;
    const double2 z = zeta[t];
    const double x = z.x - ca.zr[o], y = z.y - ca.zi[o];
    double s, c;
    sincos(x, &s, &c);
    const double ex = exp(-y);
    const double wr = 1.0 - ex * c, wi = -ex * s;          // 1 - e^{i(zeta - z_m)}
    const double v = ((t < M0) ? atan2(wi, wr) : -0.5 * log(wr * wr + wi * wi)) / (double)ca.cnt[o];
    double* row = A + (long long)t * lda + ca.off[o];
    for (int l = lane; l < ca.cnt[o]; l += 32) row[l] += v;
}

int bie_launch_add_cyl_columns(bie_ctx* ctx, int ncomp, const int32_t* counts, const int32_t* kinds, const double* zeta,
                               const double* centers, double* A, int64_t lda, cudaStream_t st)
{
    if (!ctx || !counts || !kinds || !zeta || !A) return BIE_ERR_NULL;
    if (ncomp < 1 || ncomp > BIE_MAX_COMP) return BIE_ERR_GEOMETRY;
    CylArgs ca;
    ca.nobs = 0;
    long long n = 0;
    for (int c = 0; c < ncomp; ++c) {
        if (counts[c] < 1 || kinds[c] < 0 || kinds[c] > 2 || (kinds[c] == BIE_KIND_SURFACE) != (c == 0)) return BIE_ERR_GEOMETRY;
        if (kinds[c] == BIE_KIND_OBSTACLE) {
            if (!centers) return BIE_ERR_NULL;
            ca.off[ca.nobs] = (int)n; ca.cnt[ca.nobs] = counts[c];
            ca.zr[ca.nobs] = centers[2 * ca.nobs]; ca.zi[ca.nobs] = centers[2 * ca.nobs + 1];
            ++ca.nobs;
        }
        n += counts[c];
    }
    if (n > (1 << 30)) return BIE_ERR_GEOMETRY;
    if (lda < n || (((uintptr_t)zeta) & 15u) || (((uintptr_t)A) & 7u)) return BIE_ERR_LAYOUT;
    if (ca.nobs == 0) return BIE_OK;   // no obstacle: A = B
    dim3 grid((unsigned)((n + 7) / 8), (unsigned)ca.nobs);
    bie_add_cyl_columns_kernel<<<grid, 256, 0, st>>>(ca, (int)n, counts[0], (const double2*)zeta, A, (long long)lda);
    BIE_CUDA(cudaGetLastError());
    return BIE_OK;
}
