// bie_common.cuh -- shared declarations of the CUDA path (sm_100a only).  No oracle code is shared.
//
// Pair arithmetic.  For a source node s and a target node t,
//   w = zeta_s - zeta_t = x + i y,  a = x/2,  b = y/2,
// the complex cotangent of Eq. (3.4) is assembled from PER-NODE factors, with no
// transcendental per pair:
//   S = sin(x_node/2), C = cos(x_node/2), P = exp(y_node/2), N = exp(-y_node/2)
//   sin a = S_s C_t - C_s S_t,   cos a = C_s C_t + S_s S_t
//   e^{b} = P_s N_t,  e^{-b} = N_s P_t,   D = e^b - e^-b = 2 sinh b,  G = e^b + e^-b = 2 cosh b
//   cot(w/2) = (sin a cos a - i sinh b cosh b)/(sin^2 a + sinh^2 b)
//            = (4 sin a cos a - i D G) / (4 sin^2 a + D^2)
// The assembled sin a and D cancel for |w| -> 0 (relative error about eps/|w|); pairs with
// 4 sin^2 a + D^2 < BIE_NEAR_TAU take the near path: differences first, x reduced by 2 pi, then the
// Laurent series of cot (bie_cot_half_near), which is accurate to rounding there.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/bie.h"

#define BIE_MAX_COMP 64
#define BIE_NODE_PAD 256              // node tables are padded to a multiple of the build tile width
#define BIE_NEAR_TAU 1.0e-3           // |w|^2 below which the near path is taken (|w| < 0.0316)

// SoA node table.  All double arrays have length npad.
struct NodeTable {
    const double* S;     // sin(x/2)
    const double* C;     // cos(x/2)
    const double* P;     // exp(y/2)
    const double* N;     // exp(-y/2)
    const double* QR;    // Re zeta' / (2 M_j)   (source weight)
    const double* QI;    // Im zeta' / (2 M_j)
    const double* X;     // Re zeta
    const double* Y;     // Im zeta
    const double* DIAG;  // complete diagonal entry: Im{zeta''/(2 zeta')}/M_k -+ 1/2 - EM
    const double* EM;    // [obstacle, variant A] / M_k, else 0   (E_m = M_m^{-1} e e^T)
    const int* COMP;     // component index of the node (padding: -1)
    int n;
    int npad;
};
#define BIE_NODE_ARRAYS 10

// component offsets, by value into kernels (<= 260 bytes)
struct CompTable {
    int ncomp;
    int off[BIE_MAX_COMP + 1];
};

struct bie_ctx {
    int device;
    int sm_count;
    int l2_bytes;
    int coop_ok;
    int max_smem_optin;
    // node-table storage (device), capacity in nodes
    double* node_buf;
    int* comp_buf;
    unsigned int* sync_buf;  // grid-barrier counter
    int cap;
    // current geometry (host copies)
    int have_geom;
    int n;
    int ncomp;
    int variant;
    int counts[BIE_MAX_COMP];
    int kinds[BIE_MAX_COMP];
    CompTable comps;
    // staging for bie_solve_host
    int32_t* pinned_i;  // [4]
    double* pinned_d;   // [4]
};

static inline int bie_cuda_err(cudaError_t e) { return e == cudaSuccess ? BIE_OK : BIE_ERR_CUDA_BASE - (int)e; }
#define BIE_CUDA(call)                                    \
    do {                                                  \
        cudaError_t e__ = (call);                         \
        if (e__ != cudaSuccess) return bie_cuda_err(e__); \
    } while (0)

static inline int bie_npad(int n) { return (n + BIE_NODE_PAD - 1) / BIE_NODE_PAD * BIE_NODE_PAD; }
NodeTable bie_node_table(const bie_ctx* ctx);

// internal entry points (one per .cu)
int bie_prepare_nodes(bie_ctx* ctx, int ncomp, const int32_t* counts, const int32_t* kinds,
                      const double* zeta, const double* dzeta, const double* d2zeta, int variant,
                      cudaStream_t st);
int bie_launch_build(bie_ctx* ctx, double* A, int64_t lda, int only_comp0, cudaStream_t st);
int bie_launch_matvec(bie_ctx* ctx, int n, const double* A, int64_t lda, const double* x, double* y, cudaStream_t st);
int bie_launch_matvec_free(bie_ctx* ctx, const double* x, double* y, cudaStream_t st);
int bie_launch_gmres(bie_ctx* ctx, int n, const double* A, int64_t lda, const double* rhs, double tol,
                     int restart, int max_iters, double* x, int32_t* iters_out, double* relres_out,
                     int32_t* status_out, double* res_hist, void* ws, size_t ws_bytes, cudaStream_t st);
size_t bie_gmres_ws_bytes(int n, int restart);
int bie_launch_probe_dfma(bie_ctx* ctx, int64_t fma_per_thread, double* out, int64_t* total_fma, cudaStream_t st);

// ---------------------------------------------------------------------------------------------------
// device helpers
// ---------------------------------------------------------------------------------------------------
#ifdef __CUDACC__
// 1/d for d > 0 in normal range: MUFU.RCP64H seed + two Newton steps (4 DFMA); within about 1 ulp, which
// is all an entry needs (no IEEE division sequence, no slow-path branch).  d = 0 gives inf/NaN: callers
// overwrite those pairs (s == t) afterwards.
__device__ __forceinline__ double bie_rcp(double d) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
    double e = fma(-d, r, 1.0);
    r = fma(r, e, r);
    e = fma(-d, r, 1.0);
    r = fma(r, e, r);
    return r;
}

// Near path: cot(w/2) for |w mod 2 pi| < about 0.05, from the differences x = x_s - x_t, y = y_s - y_t.
// x is reduced to (-pi, pi] with a two-word 2 pi (the kernel is 2 pi-periodic in x: the sum over images
// of Eq. (3.4)), then with z = w/2
//   cot z = 1/z - z (1/3 + z^2 (1/45 + z^2 (2/945 + z^2/4725)))      (truncation < 1e-20 |z| for |z| < 0.03)
__device__ __forceinline__ void bie_cot_half_near(double x, double y, double* re, double* im) {
    const double TWO_PI_HI = 6.283185307179586232e+00, TWO_PI_LO = 2.449293598294706414e-16;
    const double k = rint(x * 0.15915494309189534561);
    x = fma(-k, TWO_PI_HI, x);
    x = fma(-k, TWO_PI_LO, x);
    const double zr = 0.5 * x, zi = 0.5 * y;
    const double m2 = fma(zr, zr, zi * zi);
    const double inv = 1.0 / m2;
    const double z2r = fma(zr, zr, -zi * zi), z2i = 2.0 * zr * zi;
    // Horner in z^2 (complex)
    double pr = 1.0 / 4725.0, pi = 0.0, tr;
    tr = fma(pr, z2r, -pi * z2i) + 2.0 / 945.0; pi = fma(pr, z2i, pi * z2r); pr = tr;
    tr = fma(pr, z2r, -pi * z2i) + 1.0 / 45.0;  pi = fma(pr, z2i, pi * z2r); pr = tr;
    tr = fma(pr, z2r, -pi * z2i) + 1.0 / 3.0;   pi = fma(pr, z2i, pi * z2r); pr = tr;
    // 1/z - z p
    *re = zr * inv - fma(zr, pr, -zi * pi);
    *im = -zi * inv - fma(zr, pi, zi * pr);
}

__device__ __forceinline__ double bie_warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
#endif
