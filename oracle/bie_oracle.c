/*
 * bie_oracle.c -- CPU ORACLE for the boundary-integral hot path of arXiv 2108.01786.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Plain, slow, obviously-correct FP64 C written
 * from the paper; it shares no code, header, table or helper with the CUDA path
 * (paper_2108_01786_b200/csrc/).  Only tests/, __graft_entry__.smoke() and the cpu_baseline /
 * --impl reference legs of bench.py may load it.
 *
 * What it computes (every function cites the passage it follows; PAPER.md = /root/reference/PAPER.md):
 *
 *   oracle_cot_half   cot((x+iy)/2), the periodised Cauchy kernel of Eq. (3.4):
 *                     PV sum_k 1/(zeta + 2 pi k - z) = (1/2) cot((zeta - z)/2).
 *   oracle_build      the collocation matrix of Eq. (3.16), entry by entry, from
 *                     Table 1, the diagonal limit, the block
 *                     structure of Eq. (3.10), the trapezoid weights 1/M_j
 *                      and E_m = M_m^{-1} e e^T.
 *                     variant 2: the vortex-sheet system of Eqs. (4.14) + (4.17) with the adjoint
 *                     matrices K+, G+ of Eq. (4.7); its solid-solid block is Eq. (4.5).
 *   oracle_cauchy_eval   Eq. (F.4) / (5.5): a function analytic in the fluid from its boundary
 *                     values, spectrally accurate up to the boundary.
 *   oracle_add_cyl_columns   the rank-(N-1) correction of Appendix B, Eq. (B.2): stream function
 *                     prescribed on the solids, circulations unknown.
 *   oracle_normal_velocity_sums   the trapezoid sums of Eqs. (3.19) and (3.24) for the normal velocity on
 *                     Gamma_0 (Section 3.4); the FFT Hilbert transform is added in Python.
 *   oracle_matvec     y = A x, the plain definition (long-double accumulation).
 *   oracle_gmres      restarted GMRES(m) of Saad & Schultz (ref. [38] cited at PAPER.md:L855), modified
 *                     Gram-Schmidt + Givens rotations, x0 = 0, stop when the recurrence residual
 *                     |g_{j+1}| <= tol * ||b|| (PAPER.md:L869 defines i_max by this criterion).
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): P1 cot vs 40-digit mpmath and vs the image
 * sum (3.4); P2 block row sums from Eq. (6.3); P3 analytic-function reproduction; P4 spectral
 * convergence; P5 adaptive quadrature of the kernel; P6 flat/flat closed-form solution; P7 GMRES vs
 * LAPACK dgesv; P8 (variant 2) the dagger relation S = D B^T D^-1 + J against the pinned B, the Fourier
 * closed form of the flat-bottom auxiliary system, adaptive quadrature of Eq. (4.6).  Nothing here is
 * "parity unpinned".
 *
 * Readings of the paper where it is silent or garbled are listed in DESIGN.md ("Readings").
 */
#include <math.h>
#include <stdlib.h>
#define ORACLE_PI 3.14159265358979323846264338327950288
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int t)
{
#ifdef _OPENMP
    if (t > 0) omp_set_num_threads(t);
#else
    (void)t;
#endif
}

/* cot((x+iy)/2) in the half-angle form (reading R6; accuracy-critical: the form with
 * cosh y - cos x in the denominator loses 4 digits for near neighbours):
 *   cot((x+iy)/2) = ( sin(x/2)cos(x/2) - i sinh(y/2)cosh(y/2) ) / ( sin^2(x/2) + sinh^2(y/2) ).
 * 2pi-periodic in x, which is the sum over periodic images of Eq. (3.4). */
void oracle_cot_half(double x, double y, double *re, double *im)
{
    double sx = sin(0.5 * x), cx = cos(0.5 * x);
    double sh = sinh(0.5 * y), ch = cosh(0.5 * y);
    double d = sx * sx + sh * sh;
    *re = (sx * cx) / d;
    *im = -(sh * ch) / d;
}

/* One row (target node t) of the matrix of Eq. (3.16); the formulas are documented at oracle_build below.
 * comp[s] = component of node s. */
static void oracle_row(long t, long n, const int *comp, const int *counts, const int *kinds,
                       const double *zeta, const double *dzeta, const double *d2zeta, int variant, double *row)
{
    const int k = comp[t];
    const double ztr = zeta[2 * t], zti = zeta[2 * t + 1];
    for (long s = 0; s < n; ++s) {
        const int j = comp[s];
        const double Mj = (double)counts[j];
        double cre, cim;
        if (s == t) {
            /* zeta'' / (2 zeta' M) */
            double ar = d2zeta[2 * s], ai = d2zeta[2 * s + 1];
            double br = dzeta[2 * s], bi = dzeta[2 * s + 1];
            double den = br * br + bi * bi;
            cre = (ar * br + ai * bi) / den / (2.0 * Mj);
            cim = (ai * br - ar * bi) / den / (2.0 * Mj);
        } else {
            double x = zeta[2 * s] - ztr, y = zeta[2 * s + 1] - zti;
            double cr, ci;
            oracle_cot_half(x, y, &cr, &ci);
            double qr = dzeta[2 * s] / (2.0 * Mj), qi = dzeta[2 * s + 1] / (2.0 * Mj);
            cre = qr * cr - qi * ci;
            cim = qr * ci + qi * cr;
        }
        double e;
        if (k == 0 && j == 0)
            e = cim - (s == t ? 0.5 : 0.0);
        else if (k == 0)
            e = cre;
        else if (j == 0)
            e = -cre;
        else {
            e = cim + (s == t ? 0.5 : 0.0);
            if (variant == 0 && k == j && kinds[k] == 2) e -= 1.0 / Mj;
        }
        row[s] = e;
    }
}

/* One row (node t = (k,m)) of the VORTEX-SHEET system matrix S: rows on Gamma_0 are Eq. (4.14),
 * rows on solids Eq. (4.17); its trailing block (rows and columns on solids) is the matrix of
 * the auxiliary system (4.5).  The adjoint operators of Eq. (4.6) are collocated
 * with the matrices of Eq. (4.7):
 *      (K+_jk)_ml = K_jk(alpha_jl, alpha_km) / M_j,    (G+_jk)_ml = G_jk(alpha_jl, alpha_km) / M_j,
 * row m on Gamma_k, column l on Gamma_j.  With Table 1, K_jk(a,b) + i G..: the kernel's target is
 * its FIRST index, so  K_jk(alpha_jl, alpha_km) = Im c,  G_jk(alpha_jl, alpha_km) = Re c  with
 *      c = zeta'_k[m]/2 * cot((zeta_k[m] - zeta_j[l])/2)        (weight zeta' of the ROW node, argument row - column)
 * and for (k,m) == (j,l) the limit K_kk(a,a) = Im{zeta''_k/(2 zeta'_k)}.  Entry, divided by M_j:
 *      k = 0,  j = 0  :  Im c + 1/2 delta        (1/2 I + K+_00,   Eq. 4.14)
 *      k = 0,  j >= 1 : -Re c                    (-G+_j0,          Eq. 4.14)
 *      k >= 1, j = 0  :  Re c                    (G+_0k,           Eq. 4.17)
 *      k >= 1, j >= 1 :  Im c - 1/2 delta        (-1/2 I + K+_jk,  Eq. 4.5 / 4.17)                                  */
static void oracle_row_dagger(long t, long n, const int *comp, const int *counts,
                              const double *zeta, const double *dzeta, const double *d2zeta, double *row)
{
    const int k = comp[t];
    const double ztr = zeta[2 * t], zti = zeta[2 * t + 1];
    const double ur = 0.5 * dzeta[2 * t], ui = 0.5 * dzeta[2 * t + 1]; /* zeta'_k[m] / 2 */
    for (long s = 0; s < n; ++s) {
        const int j = comp[s];
        const double Mj = (double)counts[j];
        double cre, cim;
        if (s == t) {
            double ar = d2zeta[2 * s], ai = d2zeta[2 * s + 1];
            double br = dzeta[2 * s], bi = dzeta[2 * s + 1];
            double den = br * br + bi * bi;
            cre = 0.0; /* never used: G blocks have k != j */
            cim = (ai * br - ar * bi) / den / 2.0;
        } else {
            double cr, ci;
            oracle_cot_half(ztr - zeta[2 * s], zti - zeta[2 * s + 1], &cr, &ci);
            cre = ur * cr - ui * ci;
            cim = ur * ci + ui * cr;
        }
        double e;
        if (k == 0 && j == 0)
            e = cim / Mj + (s == t ? 0.5 : 0.0);
        else if (k == 0)
            e = -cre / Mj;
        else if (j == 0)
            e = cre / Mj;
        else
            e = cim / Mj - (s == t ? 0.5 : 0.0);
        row[s] = e;
    }
}

/* Matrix of Eq. (3.16).
 *
 * components: c = 0..ncomp-1 with counts[c] = M_c nodes alpha_{cl} = 2 pi l / M_c,
 * kinds[c]: 0 free surface (component 0), 1 bottom (component 1), 2 obstacle (clockwise).
 * zeta/dzeta/d2zeta: interleaved (re,im), n = sum counts, components concatenated.
 * Row = target node (k,m); column = source node (j,l).  For (k,m) != (j,l)
 *      c = zeta'_j[l] / (2 M_j) * cot((zeta_j[l] - zeta_k[m]) / 2)          (Table 1)
 * and for (k,m) == (j,l)
 *      c = zeta''_k[m] / (2 zeta'_k[m] M_k)
 * entry:  k = 0, j = 0 :  Im c - 1/2 delta          (-1/2 I + K_00)           (Eq. 3.10)
 *         k = 0, j >= 1:  Re c                      (G_0j)
 *         k >= 1, j = 0: -Re c                      (-G_k0)
 *         k >= 1, j >= 1: Im c + 1/2 delta - [k = j is an obstacle]/M_k   (1/2 I + K_kj - E_k)
 * variant 0: as above; variant 1: without the E_k term (the operator B of Eq. (3.10)); variant 2: the vortex-sheet
 * system matrix of Eqs. (4.14) + (4.17) documented at oracle_row_dagger.
 * A is row-major n x n with leading dimension lda >= n.  Returns 0, or <0 on bad arguments. */
int oracle_build(int ncomp, const int *counts, const int *kinds,
                 const double *zeta, const double *dzeta, const double *d2zeta,
                 int variant, double *A, long lda)
{
    if (ncomp < 1 || !counts || !kinds || !zeta || !dzeta || !d2zeta || !A) return -1;
    long n = 0;
    for (int c = 0; c < ncomp; ++c) {
        if (counts[c] < 1) return -2;
        if (kinds[c] < 0 || kinds[c] > 2) return -2;
        if ((kinds[c] == 0) != (c == 0)) return -2; /* the free surface is component 0, and only it */
        n += counts[c];
    }
    if (lda < n) return -3;
    int *comp = (int *)malloc(sizeof(int) * (size_t)n);
    if (!comp) return -4;
    {
        long p = 0;
        for (int c = 0; c < ncomp; ++c)
            for (int l = 0; l < counts[c]; ++l) comp[p++] = c;
    }
#pragma omp parallel for schedule(static)
    for (long t = 0; t < n; ++t) {
        if (variant == 2) oracle_row_dagger(t, n, comp, counts, zeta, dzeta, d2zeta, A + t * lda);
        else oracle_row(t, n, comp, counts, kinds, zeta, dzeta, d2zeta, variant, A + t * lda);
    }
    free(comp);
    return 0;
}

/* The listed rows of the same matrix (for sampled parity checks at sizes where the full matrix is too
 * slow): out is nrows x n, row i = row rows[i] of oracle_build's A.  Same arithmetic, same row function. */
int oracle_build_rows(int ncomp, const int *counts, const int *kinds,
                      const double *zeta, const double *dzeta, const double *d2zeta,
                      int variant, long nrows, const long *rows, double *out)
{
    if (ncomp < 1 || !counts || !kinds || !zeta || !dzeta || !d2zeta || !rows || !out) return -1;
    long n = 0;
    for (int c = 0; c < ncomp; ++c) {
        if (counts[c] < 1) return -2;
        if (kinds[c] < 0 || kinds[c] > 2) return -2;
        if ((kinds[c] == 0) != (c == 0)) return -2;
        n += counts[c];
    }
    for (long i = 0; i < nrows; ++i)
        if (rows[i] < 0 || rows[i] >= n) return -3;
    int *comp = (int *)malloc(sizeof(int) * (size_t)n);
    if (!comp) return -4;
    {
        long p = 0;
        for (int c = 0; c < ncomp; ++c)
            for (int l = 0; l < counts[c]; ++l) comp[p++] = c;
    }
#pragma omp parallel for schedule(static)
    for (long i = 0; i < nrows; ++i) {
        if (variant == 2) oracle_row_dagger(rows[i], n, comp, counts, zeta, dzeta, d2zeta, out + i * n);
        else oracle_row(rows[i], n, comp, counts, kinds, zeta, dzeta, d2zeta, variant, out + i * n);
    }
    free(comp);
    return 0;
}

/* NEXT-4, Appendix B: the variant in which the stream function is prescribed on the solids and
 * the circulation parameters a_m = <1_m, omega> are unknowns.  Eq. (B.2):
 *      A omega = B omega + sum_{m >= 2} c_m <1_m, omega>,    c_m = ( phi_cyl(zeta_0 - z_m), psi_cyl(zeta_1 - z_m), ..., psi_cyl(zeta_N - z_m) ),
 * Phi_cyl(z) = -i log(1 - e^{iz}) (Eq. (3.2)), phi_cyl = Re Phi_cyl = arg(1 - e^{iz}), psi_cyl = Im Phi_cyl =
 * -log|1 - e^{iz}|; z_m = a point inside obstacle m.  On the trapezoidal rule <1_m, omega> = (1/M_m) sum_l
 * omega_m[l], so the correction adds c_m[t]/M_m to every column of obstacle m, in every row t.
 * This function ADDS that correction to a matrix A that holds B (oracle_build with variant 1).  centers: interleaved
 * (re, im), one per component with kinds[c] == 2, in component order.  Returns 0, or < 0 on bad arguments. */
int oracle_add_cyl_columns(int ncomp, const int *counts, const int *kinds, const double *zeta, const double *centers,
                           double *A, long lda)
{
    if (ncomp < 1 || !counts || !kinds || !zeta || !A) return -1;
    long n = 0;
    for (int c = 0; c < ncomp; ++c) { if (counts[c] < 1) return -2; n += counts[c]; }
    if (lda < n) return -3;
    long off = 0;
    int o = 0;
    for (int m = 0; m < ncomp; off += counts[m], ++m) {
        if (kinds[m] != 2) continue;
        if (!centers) return -1;
        const double zr = centers[2 * o], zi = centers[2 * o + 1];
        ++o;
        const double Mm = (double)counts[m];
#pragma omp parallel for schedule(static)
        for (long t = 0; t < n; ++t) {
            /* w = 1 - e^{i(zeta_t - z_m)} */
            const double x = zeta[2 * t] - zr, y = zeta[2 * t + 1] - zi;
            const double ex = exp(-y);
            const double wr = 1.0 - ex * cos(x), wi = -ex * sin(x);
            const double c = (t < counts[0]) ? atan2(wi, wr) : -0.5 * log(wr * wr + wi * wi);
            for (long l = 0; l < counts[m]; ++l) A[t * lda + off + l] += c / Mm;
        }
    }
    return 0;
}

/* NEXT-3, Section 5.1 / Appendix F: evaluation of a function analytic in the fluid from
 * its boundary values, spectrally accurate up to the boundary (Helsing & Ojala, periodic version).  Eq. (F.4) / (5.5):
 *      f(z) ~ sum_km lambda~_km(z) f(zeta_k(alpha_m)) / sum_km lambda~_km(z),
 *      lambda~_km(z) = (sigma_k / M_k) * 1/2 cot((zeta_k(alpha_m) - z)/2) * zeta'_k(alpha_m),
 * with sigma_0 = -1 and sigma_k = +1 for the solids: Gamma_0 is parameterised with the fluid on its RIGHT, so it
 * enters the boundary integral of (F.1) with the opposite orientation (reading R18; (F.3)/(F.4) do not print it).
 * "If z coincides with zeta_k(alpha_m), we set f(z) = f(zeta_k(alpha_m))".
 * f: nf functions, [nf][n] complex interleaved; zpts: npts complex; out: [nf][npts] complex.  Returns 0 or < 0. */
int oracle_cauchy_eval(int ncomp, const int *counts, const int *kinds, const double *zeta, const double *dzeta,
                       int nf, const double *f, long npts, const double *zpts, double *out)
{
    if (ncomp < 1 || !counts || !kinds || !zeta || !dzeta || !f || !zpts || !out || nf < 1) return -1;
    long n = 0;
    for (int c = 0; c < ncomp; ++c) { if (counts[c] < 1) return -2; n += counts[c]; }
#pragma omp parallel for schedule(static)
    for (long p = 0; p < npts; ++p) {
        const double zr = zpts[2 * p], zi = zpts[2 * p + 1];
        long double Dr = 0.0L, Di = 0.0L;
        long double Nr[8], Ni[8];
        for (int q = 0; q < nf && q < 8; ++q) { Nr[q] = 0.0L; Ni[q] = 0.0L; }
        long hit = -1;
        long s = 0;
        for (int k = 0; k < ncomp && hit < 0; ++k) {
            const double wgt = (kinds[k] == 0 ? -1.0 : 1.0) / (double)counts[k];
            for (long m = 0; m < counts[k]; ++m, ++s) {
                const double x = zeta[2 * s] - zr, y = zeta[2 * s + 1] - zi;
                const double sx = sin(0.5 * x), sh = sinh(0.5 * y);
                if (sx * sx + sh * sh == 0.0) { hit = s; break; }
                double cr, ci;
                oracle_cot_half(x, y, &cr, &ci);
                /* lambda~ = wgt * 1/2 * cot * zeta' */
                const double lr = 0.5 * wgt * (cr * dzeta[2 * s] - ci * dzeta[2 * s + 1]);
                const double li = 0.5 * wgt * (cr * dzeta[2 * s + 1] + ci * dzeta[2 * s]);
                Dr += lr; Di += li;
                for (int q = 0; q < nf && q < 8; ++q) {
                    const double fr = f[2 * ((long)q * n + s)], fi = f[2 * ((long)q * n + s) + 1];
                    Nr[q] += (long double)lr * fr - (long double)li * fi;
                    Ni[q] += (long double)lr * fi + (long double)li * fr;
                }
            }
        }
        for (int q = 0; q < nf && q < 8; ++q) {
            double *o = out + 2 * ((long)q * npts + p);
            if (hit >= 0) { o[0] = f[2 * ((long)q * n + hit)]; o[1] = f[2 * ((long)q * n + hit) + 1]; }
            else {
                const long double d2 = Dr * Dr + Di * Di;
                o[0] = (double)((Nr[q] * Dr + Ni[q] * Di) / d2);
                o[1] = (double)((Ni[q] * Dr - Nr[q] * Di) / d2);
            }
        }
    }
    return nf > 8 ? -5 : 0;
}

/* NEXT-2: the trapezoid sums of the normal velocity on the free surface, Section 3.4, for the
 * listed nodes m of Gamma_0 (component 0).  With w = omega' (the derivatives of the densities, all components
 * concatenated) the function returns, per listed node,
 *      out = - (1/M_0) sum_l G_00(alpha_l, alpha_m) w_0[l]  +  sum_{j>=1} (1/M_j) sum_l K_j0(alpha_jl, alpha_m) w_j[l],
 * i.e. the integral of Eq. (3.24) and the integrals of Eq. (3.19) on the
 * trapezoidal rule ("which we evaluate with spectral accuracy using the trapezoidal rule").  The
 * integration variable is in the FIRST slot of the kernels: with Table 1
 *      K_j0(beta, alpha) = Im{ zeta'_0(alpha)/2 cot((zeta_0(alpha) - zeta_j(beta))/2) },
 *      G_00(beta, alpha) = Re{ zeta'_0(alpha)/2 cot((zeta_0(alpha) - zeta_0(beta))/2) } - 1/2 cot((alpha - beta)/2),
 * and G_00(alpha, alpha) = Re{zeta''_0/(2 zeta'_0)} (the bracket of Eq. (3.23) tends to -zeta''/(2 zeta')).
 * The Hilbert-transform term -1/2 H omega'_0 of Eq. (3.24) and the phi_mv term (3.17) are NOT included here: the
 * caller adds them (FFT, symbol -i sgn k).  Returns 0, or < 0 on bad arguments. */
int oracle_normal_velocity_sums(int ncomp, const int *counts, const double *zeta, const double *dzeta,
                                const double *d2zeta, const double *w, long nrows, const long *rows, double *out)
{
    if (ncomp < 1 || !counts || !zeta || !dzeta || !d2zeta || !w || !rows || !out) return -1;
    long n = 0;
    for (int c = 0; c < ncomp; ++c) { if (counts[c] < 1) return -2; n += counts[c]; }
    const long M0 = counts[0];
    for (long i = 0; i < nrows; ++i) if (rows[i] < 0 || rows[i] >= M0) return -3;
#pragma omp parallel for schedule(static)
    for (long i = 0; i < nrows; ++i) {
        const long m = rows[i];
        const double ur = 0.5 * dzeta[2 * m], ui = 0.5 * dzeta[2 * m + 1]; /* zeta'_0(alpha_m)/2 */
        const double alpha_m = 2.0 * ORACLE_PI * (double)m / (double)M0;
        long double acc = 0.0L;
        long s = 0;
        for (int j = 0; j < ncomp; ++j) {
            const double Mj = (double)counts[j];
            for (long l = 0; l < counts[j]; ++l, ++s) {
                double e;
                if (s == m) { /* j = 0, beta = alpha: G_00(alpha, alpha) */
                    double ar = d2zeta[2 * s], ai = d2zeta[2 * s + 1], br = dzeta[2 * s], bi = dzeta[2 * s + 1];
                    e = -((ar * br + ai * bi) / (br * br + bi * bi)) / 2.0;
                } else {
                    double cr, ci;
                    oracle_cot_half(zeta[2 * m] - zeta[2 * s], zeta[2 * m + 1] - zeta[2 * s + 1], &cr, &ci);
                    const double cre = ur * cr - ui * ci, cim = ur * ci + ui * cr;
                    if (j == 0) {
                        const double beta_l = 2.0 * ORACLE_PI * (double)l / (double)M0;
                        e = -(cre - 0.5 / tan(0.5 * (alpha_m - beta_l)));
                    } else {
                        e = cim;
                    }
                }
                acc += (long double)(e / Mj) * (long double)w[s];
            }
        }
        out[i] = (double)acc;
    }
    return 0;
}

/* y = A x for a rectangular nrows x ncols block, plain definition, long-double accumulation so the
 * oracle is the more accurate side. */
void oracle_matvec_rect(long nrows, long ncols, const double *A, long lda, const double *x, double *y)
{
#pragma omp parallel for schedule(static)
    for (long i = 0; i < nrows; ++i) {
        const double *row = A + i * lda;
        long double acc = 0.0L;
        for (long j = 0; j < ncols; ++j) acc += (long double)row[j] * (long double)x[j];
        y[i] = (double)acc;
    }
}

/* y = A x, square. */
void oracle_matvec(long n, const double *A, long lda, const double *x, double *y)
{
    oracle_matvec_rect(n, n, A, lda, x, y);
}

static double dot_ld(long n, const double *a, const double *b)
{
    long double acc = 0.0L;
    for (long i = 0; i < n; ++i) acc += (long double)a[i] * (long double)b[i];
    return (double)acc;
}

/* Restarted GMRES(m), Saad-Schultz (ref. [38]), unpreconditioned, on the unscaled
 * system (3.16); readings R8-R10:
 *   1. x = 0, bn = ||b||, iters = 0.
 *   2. cycle: r = b - A x (first cycle r = b); beta = ||r||; stop if beta <= tol bn.
 *      v_1 = r / beta, g = beta e_1.
 *   3. j = 1..m: w = A v_j; modified Gram-Schmidt against v_1..v_j -> h_{1..j,j};
 *      h_{j+1,j} = ||w||; v_{j+1} = w / h_{j+1,j}; apply rotations 1..j-1 to column j; rotation j from
 *      (h_jj, h_{j+1,j}) with d = hypot; g_{j+1} = -s_j g_j, g_j = c_j g_j; iters += 1;
 *      leave the loop when |g_{j+1}| <= tol bn   (i_max of PAPER.md:L869 counts these steps).
 *   4. y = R^{-1} g, x += sum y_i v_i; converged -> stop, else restart at 2.
 * Outputs: x, *iters, *relres = ||b - A x|| / bn (true residual; reported, never used to continue),
 * res_hist[i] (i = 0..iters; optional) = recurrence residual / bn after i steps.
 * Returns 0 converged, 1 max_iters reached, <0 bad arguments. */
int oracle_gmres(long n, const double *A, long lda, const double *b,
                 double tol, int restart, int max_iters,
                 double *x, int *iters_out, double *relres_out, double *res_hist)
{
    if (n < 1 || !A || !b || !x || restart < 1 || max_iters < 0 || lda < n) return -1;
    const int m = restart;
    double *V = (double *)malloc(sizeof(double) * (size_t)(m + 1) * (size_t)n);
    double *H = (double *)calloc((size_t)(m + 1) * (size_t)m, sizeof(double)); /* H[i + j*(m+1)] */
    double *cs = (double *)malloc(sizeof(double) * (size_t)m);
    double *sn = (double *)malloc(sizeof(double) * (size_t)m);
    double *g = (double *)malloc(sizeof(double) * (size_t)(m + 1));
    double *w = (double *)malloc(sizeof(double) * (size_t)n);
    double *yv = (double *)malloc(sizeof(double) * (size_t)m);
    if (!V || !H || !cs || !sn || !g || !w || !yv) {
        free(V); free(H); free(cs); free(sn); free(g); free(w); free(yv);
        return -4;
    }
    for (long i = 0; i < n; ++i) x[i] = 0.0;
    const double bn = sqrt(dot_ld(n, b, b));
    int iters = 0, converged = 0, first = 1;
    if (res_hist) res_hist[0] = 1.0;
    if (bn == 0.0) converged = 1;
    while (!converged && iters < max_iters) {
        /* step 2 */
        if (first) {
            memcpy(w, b, sizeof(double) * (size_t)n);
            first = 0;
        } else {
            oracle_matvec(n, A, lda, x, w);
            for (long i = 0; i < n; ++i) w[i] = b[i] - w[i];
        }
        double beta = sqrt(dot_ld(n, w, w));
        if (beta <= tol * bn) { converged = 1; break; }
        for (long i = 0; i < n; ++i) V[i] = w[i] / beta;
        g[0] = beta;
        int k = 0;
        /* step 3 */
        for (int j = 0; j < m && iters < max_iters; ++j) {
            double *vj = V + (size_t)j * (size_t)n;
            oracle_matvec(n, A, lda, vj, w);
            double *hcol = H + (size_t)j * (size_t)(m + 1);
            for (int i = 0; i <= j; ++i) {
                const double *vi = V + (size_t)i * (size_t)n;
                double h = dot_ld(n, vi, w);
                hcol[i] = h;
                for (long r = 0; r < n; ++r) w[r] -= h * vi[r];
            }
            double hn = sqrt(dot_ld(n, w, w));
            hcol[j + 1] = hn;
            if (hn != 0.0) {
                double *vn = V + (size_t)(j + 1) * (size_t)n;
                for (long r = 0; r < n; ++r) vn[r] = w[r] / hn;
            }
            for (int i = 0; i < j; ++i) {
                double t0 = cs[i] * hcol[i] + sn[i] * hcol[i + 1];
                double t1 = -sn[i] * hcol[i] + cs[i] * hcol[i + 1];
                hcol[i] = t0;
                hcol[i + 1] = t1;
            }
            double d = hypot(hcol[j], hcol[j + 1]);
            if (d == 0.0) { cs[j] = 1.0; sn[j] = 0.0; }
            else { cs[j] = hcol[j] / d; sn[j] = hcol[j + 1] / d; }
            hcol[j] = d;
            hcol[j + 1] = 0.0;
            g[j + 1] = -sn[j] * g[j];
            g[j] = cs[j] * g[j];
            ++iters;
            k = j + 1;
            if (res_hist) res_hist[iters] = fabs(g[j + 1]) / bn;
            if (fabs(g[j + 1]) <= tol * bn || hn == 0.0) { converged = 1; break; }
        }
        /* step 4: back-substitution R y = g (size k), x += V y */
        for (int i = k - 1; i >= 0; --i) {
            double s = g[i];
            for (int c = i + 1; c < k; ++c) s -= H[(size_t)c * (size_t)(m + 1) + i] * yv[c];
            yv[i] = s / H[(size_t)i * (size_t)(m + 1) + i];
        }
        for (int i = 0; i < k; ++i) {
            const double *vi = V + (size_t)i * (size_t)n;
            const double yi = yv[i];
            for (long r = 0; r < n; ++r) x[r] += yi * vi[r];
        }
    }
    /* true residual */
    double relres = 0.0;
    if (bn != 0.0) {
        oracle_matvec(n, A, lda, x, w);
        for (long i = 0; i < n; ++i) w[i] = b[i] - w[i];
        relres = sqrt(dot_ld(n, w, w)) / bn;
    }
    if (iters_out) *iters_out = iters;
    if (relres_out) *relres_out = relres;
    free(V); free(H); free(cs); free(sn); free(g); free(w); free(yv);
    return converged ? 0 : 1;
}
