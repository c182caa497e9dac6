// bie_noalloc.cu -- bie_gmres_noalloc (include/bie.h): the stored-matrix GMRES solve for callers that cannot call
// cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).  The workspace the solve
// needs (Krylov basis, per-CTA partials, R, y, the grid-barrier counter: bie_gmres.cu, gmres_ws_layout) lives in ONE
// file-scope device array of BIE_NOALLOC_SCRATCH_BYTES that every GPU loading the library holds until exit.  The kernel
// is the one bie_gmres launches; it receives the array's DEVICE address as its workspace pointer.
//
// In host code the array's name is a host-side stand-in, not a device address: the address comes from
// cudaGetSymbolAddress, looked up once per device with that device current (first call on the device, or
// bie_gmres_noalloc on any later call finds it cached).  Nothing here calls cudaMalloc, cudaFree or an allocating
// library routine.
#include <mutex>
#include "bie_common.cuh"

static __device__ __align__(256) unsigned char g_noalloc_scratch[BIE_NOALLOC_SCRATCH_BYTES];

#define BIE_NOALLOC_MAX_DEVICES 64
static void* g_scratch_ptr[BIE_NOALLOC_MAX_DEVICES];   // device address of g_noalloc_scratch on device i (0: not looked up yet)
static std::mutex g_scratch_mutex;

// the device address of the scratch array on `device`, which must be current
static int noalloc_scratch(int device, void** out)
{
    if (device < 0 || device >= BIE_NOALLOC_MAX_DEVICES) return BIE_ERR_DEVICE;
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_ptr[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess) { cudaGetLastError(); return bie_cuda_err(e); }
        if (!p || (((uintptr_t)p) & 255u)) return BIE_ERR_LAYOUT;
        g_scratch_ptr[device] = p;
    }
    *out = g_scratch_ptr[device];
    return BIE_OK;
}

extern "C" {

size_t bie_gmres_noalloc_max_bytes(void) { return (size_t)BIE_NOALLOC_SCRATCH_BYTES; }

int bie_gmres_noalloc(bie_ctx* c, int n, const double* A, int64_t lda, const double* rhs, double tol, int restart,
                      int max_iters, double* x, int32_t* iters_out, double* relres_out, int32_t* status_out,
                      void* stream)
{
    if (!c || !A) return BIE_ERR_NULL;                       // stored matrix only: the matrix-free operator's near matrix allocates
    if (n < 1 || restart < 1) return BIE_ERR_ARG;
    // sizes beyond the static scratch are rejected before anything is launched
    const size_t need = bie_gmres_ws_bytes(n, restart);
    if (need == 0 || need > (size_t)BIE_NOALLOC_SCRATCH_BYTES) return BIE_ERR_NOALLOC_SIZE;
    BIE_CUDA(cudaSetDevice(c->device));
    void* ws = nullptr;
    const int rc = noalloc_scratch(c->device, &ws);
    if (rc != BIE_OK) return rc;
    // the array keeps the last call's contents: the solve writes every part of its workspace before reading it, except
    // the grid-barrier counter, which bie_launch_gmres clears on the stream before the launch
    return bie_launch_gmres(c, n, A, lda, 0, rhs, tol, restart, max_iters, x, iters_out, relres_out, status_out, nullptr,
                            ws, (size_t)BIE_NOALLOC_SCRATCH_BYTES, (cudaStream_t)stream);
}

}  // extern "C"
