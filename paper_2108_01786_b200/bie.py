"""Thin Python binding of the C-ABI library (include/bie.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of ``csrc/``; PyTorch supplies device memory and streams.
There is no CPU fallback: ``lib()`` raises if ``libbie_b200.so`` is missing, ``Context()`` raises unless a
compute-capability-10.x device is present.  Nothing here imports ``oracle``.

Names follow the header: bie_build, bie_build_update, bie_set_geometry, bie_matvec, bie_matvec_free,
bie_gmres, bie_solve_host, bie_probe_dfma.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbie_b200.so")
_lib: Optional[ctypes.CDLL] = None

# the symbols include/bie.h declares
EXPORTS = ("bie_create", "bie_destroy", "bie_strerror", "bie_device_info", "bie_build", "bie_build_update",
           "bie_set_geometry", "bie_matvec", "bie_matvec_free", "bie_gmres_workspace_bytes", "bie_gmres",
           "bie_solve_workspace_bytes", "bie_solve_host", "bie_probe_dfma", "bie_build_cols", "bie_hybrid_cols",
           "bie_set_hybrid_free_warps", "bie_gmres_hybrid", "bie_matvec_rect", "bie_build_normal_velocity",
           "bie_add_cyl_columns", "bie_cauchy_eval_workspace_bytes", "bie_cauchy_eval", "bie_set_symmetric",
           "bie_build_block", "bie_set_hybrid_poll_tiles", "bie_hybrid_block_bytes", "bie_probe_read",
           "bie_gmres_noalloc", "bie_gmres_noalloc_max_bytes", "bie_set_small_gmres")

BIE_OK, BIE_MAX_ITERS = 0, 1
OP_DENSE, OP_FREE, OP_HYBRID = 0, 1, 2
VARIANT_A, VARIANT_B, VARIANT_VORTEX = 0, 1, 2


class BieError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {strerror(code)} (code {code})")


def lib() -> ctypes.CDLL:
    """Loads libbie_b200.so (built by ``python -m paper_2108_01786_b200.build``).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2108_01786_b200.build` "
                              "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, i32, i64, dbl, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_double, ctypes.c_size_t
        ip = ctypes.POINTER(ctypes.c_int32)
        L.bie_create.restype = i32
        L.bie_create.argtypes = [ctypes.POINTER(vp), i32]
        L.bie_destroy.restype = i32
        L.bie_destroy.argtypes = [vp]
        L.bie_strerror.restype = ctypes.c_char_p
        L.bie_strerror.argtypes = [i32]
        L.bie_device_info.restype = i32
        L.bie_device_info.argtypes = [vp, ip, ip, ip]
        geo = [vp, i32, ip, ip, vp, vp, vp, i32]
        L.bie_build.restype = i32
        L.bie_build.argtypes = geo + [vp, i64, vp]
        L.bie_build_update.restype = i32
        L.bie_build_update.argtypes = geo + [vp, i64, vp]
        L.bie_set_geometry.restype = i32
        L.bie_set_geometry.argtypes = geo + [vp]
        L.bie_matvec.restype = i32
        L.bie_matvec.argtypes = [vp, i32, vp, i64, vp, vp, vp]
        L.bie_matvec_free.restype = i32
        L.bie_matvec_free.argtypes = [vp, i32, vp, vp, vp]
        L.bie_gmres_workspace_bytes.restype = sz
        L.bie_gmres_workspace_bytes.argtypes = [i32, i32]
        L.bie_gmres.restype = i32
        L.bie_gmres.argtypes = [vp, i32, vp, i64, vp, dbl, i32, i32, vp, vp, vp, vp, vp, vp, sz, vp]
        L.bie_gmres_noalloc.restype = i32
        L.bie_gmres_noalloc.argtypes = [vp, i32, vp, i64, vp, dbl, i32, i32, vp, vp, vp, vp, vp]
        L.bie_gmres_noalloc_max_bytes.restype = sz
        L.bie_gmres_noalloc_max_bytes.argtypes = []
        L.bie_solve_workspace_bytes.restype = sz
        L.bie_solve_workspace_bytes.argtypes = [i32, i32, i32]
        L.bie_solve_host.restype = i32
        L.bie_solve_host.argtypes = [vp, i32, ip, ip, vp, vp, vp, vp, dbl, i32, i32, i32, vp, ip,
                                     ctypes.POINTER(dbl), vp, sz, vp]
        L.bie_build_cols.restype = i32
        L.bie_build_cols.argtypes = geo + [i32, vp, i64, vp]
        L.bie_build_block.restype = i32
        L.bie_build_block.argtypes = geo + [i32, vp, vp]
        L.bie_hybrid_block_bytes.restype = sz
        L.bie_hybrid_block_bytes.argtypes = [i32]
        L.bie_hybrid_cols.restype = i32
        L.bie_hybrid_cols.argtypes = [vp, i32]
        L.bie_set_hybrid_free_warps.restype = i32
        L.bie_set_hybrid_free_warps.argtypes = [vp, i32]
        L.bie_set_hybrid_poll_tiles.restype = i32
        L.bie_set_hybrid_poll_tiles.argtypes = [vp, i32]
        L.bie_gmres_hybrid.restype = i32
        L.bie_gmres_hybrid.argtypes = [vp, i32, vp, i32, vp, dbl, i32, i32, vp, vp, vp, vp, vp, vp, sz, vp]
        L.bie_matvec_rect.restype = i32
        L.bie_matvec_rect.argtypes = [vp, i32, i32, vp, i64, vp, vp, vp]
        L.bie_build_normal_velocity.restype = i32
        L.bie_build_normal_velocity.argtypes = geo[:-1] + [vp, i64, vp]
        L.bie_add_cyl_columns.restype = i32
        L.bie_add_cyl_columns.argtypes = [vp, i32, ip, ip, vp, ctypes.POINTER(dbl), vp, i64, vp]
        L.bie_cauchy_eval_workspace_bytes.restype = sz
        L.bie_cauchy_eval_workspace_bytes.argtypes = [vp, i32, i32]
        L.bie_cauchy_eval.restype = i32
        L.bie_cauchy_eval.argtypes = [vp, i32, ip, ip, vp, vp, i32, vp, i32, vp, vp, vp, sz, vp]
        L.bie_set_symmetric.restype = i32
        L.bie_set_symmetric.argtypes = [vp, i32]
        L.bie_set_small_gmres.restype = i32
        L.bie_set_small_gmres.argtypes = [vp, i32]
        L.bie_probe_read.restype = i32
        L.bie_probe_read.argtypes = [vp, vp, i64, vp, vp]
        L.bie_probe_dfma.restype = i32
        L.bie_probe_dfma.argtypes = [vp, i64, vp, ctypes.POINTER(i64), vp]
        _lib = L
    return _lib


def strerror(code: int) -> str:
    return lib().bie_strerror(int(code)).decode()


def _check(rc: int, where: str, ok=(BIE_OK,)) -> int:
    if rc not in ok:
        raise BieError(rc, where)
    return rc


def _stream() -> int:
    import torch
    return int(torch.cuda.current_stream().cuda_stream)


def _i32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int32)


def _ip(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))


def _dev_c128(t, n: int) -> int:
    """device pointer of a complex128 (or interleaved float64 [n,2]) CUDA tensor of n nodes"""
    import torch
    assert t.is_cuda and t.is_contiguous()
    assert (t.dtype == torch.complex128 and t.numel() == n) or (t.dtype == torch.float64 and t.numel() == 2 * n)
    return t.data_ptr()


def _dev_f64(t, nmin: int) -> int:
    import torch
    assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.numel() >= nmin
    return t.data_ptr()


class Context:
    """Owns a ``bie_ctx`` (node tables of the current geometry, barrier counter).  One per stream."""

    def __init__(self, device: int = 0):
        self._h = ctypes.c_void_p()
        _check(lib().bie_create(ctypes.byref(self._h), int(device)), "bie_create")
        self.device = int(device)
        sm, fma, l2 = ctypes.c_int32(), ctypes.c_int32(), ctypes.c_int32()
        _check(lib().bie_device_info(self._h, ctypes.byref(sm), ctypes.byref(fma), ctypes.byref(l2)), "bie_device_info")
        self.sm_count, self.fp64_fma_per_sm_clk, self.l2_mib = sm.value, fma.value, l2.value

    def close(self):
        if self._h:
            lib().bie_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- (a) build ---------------------------------------------------------------------------------
    def _geo(self, counts, kinds, zeta, dzeta, d2zeta, variant):
        counts, kinds = _i32(counts), _i32(kinds)
        n = int(counts.sum())
        return n, [self._h, int(counts.size), _ip(counts), _ip(kinds), _dev_c128(zeta, n), _dev_c128(dzeta, n),
                   _dev_c128(d2zeta, n), int(variant)], (counts, kinds)

    def bie_build(self, counts, kinds, zeta, dzeta, d2zeta, A, variant: int = VARIANT_A, lda: Optional[int] = None):
        """A (CUDA float64, n x lda row-major) <- matrix of Eq. (3.16); returns A."""
        n, args, keep = self._geo(counts, kinds, zeta, dzeta, d2zeta, variant)
        lda = int(lda if lda is not None else A.stride(0))
        _dev_f64(A, (n - 1) * lda + n)
        _check(lib().bie_build(*args, A.data_ptr(), lda, _stream()), "bie_build")
        return A

    def bie_build_update(self, counts, kinds, zeta, dzeta, d2zeta, A, variant: int = VARIANT_A,
                         lda: Optional[int] = None):
        n, args, keep = self._geo(counts, kinds, zeta, dzeta, d2zeta, variant)
        lda = int(lda if lda is not None else A.stride(0))
        _dev_f64(A, (n - 1) * lda + n)
        _check(lib().bie_build_update(*args, A.data_ptr(), lda, _stream()), "bie_build_update")
        return A

    def bie_build_cols(self, counts, kinds, zeta, dzeta, d2zeta, ncols: int, A, variant: int = VARIANT_A,
                       lda: Optional[int] = None):
        """A (CUDA float64, n x lda row-major, lda >= ncols) <- columns [0, ncols) of the matrix of Eq. (3.16)
        (all n rows; the hybrid operator reads only the leading ncols x ncols block of it, see bie_build_block)."""
        n, args, keep = self._geo(counts, kinds, zeta, dzeta, d2zeta, variant)
        lda = int(lda if lda is not None else A.stride(0))
        _dev_f64(A, (n - 1) * lda + int(ncols))
        _check(lib().bie_build_cols(*args, int(ncols), A.data_ptr(), lda, _stream()), "bie_build_cols")
        return A

    @staticmethod
    def bie_hybrid_block_bytes(nblock: int) -> int:
        return int(lib().bie_hybrid_block_bytes(int(nblock)))

    def bie_build_block(self, counts, kinds, zeta, dzeta, d2zeta, nblock: int, A, variant: int = VARIANT_A):
        """A (CUDA float64, bie_hybrid_block_bytes(nblock) bytes) <- the leading nblock x nblock block of the matrix in the
        library's block format (tiles of 4 x 512, each contiguous): the stored part of the hybrid operator."""
        n, args, keep = self._geo(counts, kinds, zeta, dzeta, d2zeta, variant)
        _dev_f64(A, self.bie_hybrid_block_bytes(nblock) // 8)
        _check(lib().bie_build_block(*args, int(nblock), A.data_ptr(), _stream()), "bie_build_block")
        return A

    def bie_hybrid_cols(self, n: int) -> int:
        return int(lib().bie_hybrid_cols(self._h, int(n)))

    def bie_set_hybrid_free_warps(self, free_warps: int):
        _check(lib().bie_set_hybrid_free_warps(self._h, int(free_warps)), "bie_set_hybrid_free_warps")

    def bie_set_hybrid_poll_tiles(self, tiles: int):
        _check(lib().bie_set_hybrid_poll_tiles(self._h, int(tiles)), "bie_set_hybrid_poll_tiles")

    def bie_set_geometry(self, counts, kinds, zeta, dzeta, d2zeta, variant: int = VARIANT_A):
        n, args, keep = self._geo(counts, kinds, zeta, dzeta, d2zeta, variant)
        _check(lib().bie_set_geometry(*args, _stream()), "bie_set_geometry")

    # ---- (b) matvec --------------------------------------------------------------------------------
    def bie_matvec(self, A, x, y, lda: Optional[int] = None):
        n = x.numel()
        lda = int(lda if lda is not None else A.stride(0))
        _check(lib().bie_matvec(self._h, n, _dev_f64(A, (n - 1) * lda + n), lda, _dev_f64(x, n), _dev_f64(y, n),
                                _stream()), "bie_matvec")
        return y

    def bie_matvec_rect(self, A, x, y, lda: Optional[int] = None):
        """y (nrows = y.numel()) = A (nrows x ncols, ncols = x.numel()) x"""
        nrows, ncols = y.numel(), x.numel()
        lda = int(lda if lda is not None else A.stride(0))
        _check(lib().bie_matvec_rect(self._h, nrows, ncols, _dev_f64(A, (nrows - 1) * lda + ncols), lda, _dev_f64(x, ncols),
                                     _dev_f64(y, nrows), _stream()), "bie_matvec_rect")
        return y

    def bie_build_normal_velocity(self, counts, kinds, zeta, dzeta, d2zeta, Nmat, lda: Optional[int] = None):
        """Nmat (CUDA float64, M_0 x lda, lda >= n) <- the normal-velocity operator of Section 3.4 (Eqs. 3.19 + 3.24)."""
        n, args, keep = self._geo(counts, kinds, zeta, dzeta, d2zeta, 0)
        M0 = int(keep[0][0])
        lda = int(lda if lda is not None else Nmat.stride(0))
        _dev_f64(Nmat, (M0 - 1) * lda + n)
        _check(lib().bie_build_normal_velocity(*args[:-1], Nmat.data_ptr(), lda, _stream()), "bie_build_normal_velocity")
        return Nmat

    def bie_add_cyl_columns(self, counts, kinds, zeta, centers, A, lda: Optional[int] = None):
        """A (holding the operator B, variant 1) += the correction columns of Appendix B, Eq. (B.2); centers: one complex
        point per obstacle (host)."""
        counts, kinds = _i32(counts), _i32(kinds)
        n = int(counts.sum())
        zc = np.ascontiguousarray(np.asarray(centers, dtype=np.complex128).reshape(-1))
        zf = zc.view(np.float64) if zc.size else np.zeros(2)
        lda = int(lda if lda is not None else A.stride(0))
        _check(lib().bie_add_cyl_columns(self._h, int(counts.size), _ip(counts), _ip(kinds), _dev_c128(zeta, n),
                                         zf.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                                         _dev_f64(A, (n - 1) * lda + n), lda, _stream()), "bie_add_cyl_columns")
        return A

    def bie_cauchy_eval(self, counts, kinds, zeta, dzeta, fvals, zpts, out=None):
        """Eq. (F.4)/(5.5): fvals (CUDA complex128, nf x n) at the boundary nodes -> values at zpts (CUDA complex128, npts);
        returns out (nf x npts complex128)."""
        import torch
        counts, kinds = _i32(counts), _i32(kinds)
        n = int(counts.sum())
        fv = fvals if fvals.dim() == 2 else fvals[None, :]
        nf, npts = int(fv.shape[0]), int(zpts.numel())
        assert fv.is_cuda and fv.dtype == torch.complex128 and fv.is_contiguous() and fv.shape[1] == n
        assert zpts.is_cuda and zpts.dtype == torch.complex128 and zpts.is_contiguous()
        if out is None:
            out = torch.empty((nf, npts), dtype=torch.complex128, device=zpts.device)
        ws = torch.empty(int(lib().bie_cauchy_eval_workspace_bytes(self._h, nf, npts)), dtype=torch.uint8, device=zpts.device)
        _check(lib().bie_cauchy_eval(self._h, int(counts.size), _ip(counts), _ip(kinds), _dev_c128(zeta, n), _dev_c128(dzeta, n),
                                     nf, fv.data_ptr(), npts, zpts.data_ptr(), out.data_ptr(), ws.data_ptr(), ws.numel(),
                                     _stream()), "bie_cauchy_eval")
        return out

    def bie_set_small_gmres(self, on):
        """1 (default): stored-matrix solves up to n = 640 run on one thread-block cluster (bie_gmres_cluster.cu); 0: always the grid-wide kernel"""
        _check(lib().bie_set_small_gmres(self._h, int(on)), "bie_set_small_gmres")

    def bie_set_symmetric(self, on):
        """0: one-directional pair loops; 1 (default): symmetric loops in the whole-matrix matrix-free operator; 2: also in
        the hybrid operator"""
        _check(lib().bie_set_symmetric(self._h, int(on)), "bie_set_symmetric")

    def bie_matvec_free(self, x, y):
        n = x.numel()
        _check(lib().bie_matvec_free(self._h, n, _dev_f64(x, n), _dev_f64(y, n), _stream()), "bie_matvec_free")
        return y

    # ---- (c) GMRES ---------------------------------------------------------------------------------
    @staticmethod
    def bie_gmres_workspace_bytes(n: int, restart: int) -> int:
        return int(lib().bie_gmres_workspace_bytes(int(n), int(restart)))

    def bie_gmres(self, A, rhs, x, tol: float, restart: int, max_iters: int, workspace, out_i32, out_f64,
                  lda: Optional[int] = None, res_hist=None):
        """Asynchronous.  A = None selects the matrix-free operator.  out_i32: CUDA int32[2] <- (iters, status);
        out_f64: CUDA float64[1] <- true relative residual; res_hist: optional CUDA float64[max_iters+1]."""
        import torch
        n = rhs.numel()
        if A is None:
            pA, lda = None, 0
        else:
            lda = int(lda if lda is not None else A.stride(0))
            pA = _dev_f64(A, (n - 1) * lda + n)
        assert out_i32.is_cuda and out_i32.dtype == torch.int32 and out_i32.numel() >= 2
        assert workspace.is_cuda and workspace.is_contiguous()
        ws_bytes = workspace.numel() * workspace.element_size()
        _check(lib().bie_gmres(self._h, n, pA, lda, _dev_f64(rhs, n), float(tol), int(restart), int(max_iters),
                               _dev_f64(x, n), out_i32.data_ptr(), _dev_f64(out_f64, 1),
                               out_i32.data_ptr() + 4,
                               None if res_hist is None else _dev_f64(res_hist, int(max_iters) + 1),
                               workspace.data_ptr(), ws_bytes, _stream()), "bie_gmres")
        return x

    @staticmethod
    def bie_gmres_noalloc_max_bytes() -> int:
        return int(lib().bie_gmres_noalloc_max_bytes())

    def bie_gmres_noalloc(self, A, rhs, x, tol: float, restart: int, max_iters: int, out_i32, out_f64,
                          lda: Optional[int] = None):
        """Asynchronous.  bie_gmres with the stored matrix A and NO workspace argument: the workspace is a static device
        array inside the library (bie_gmres_workspace_bytes(n, restart) must not exceed bie_gmres_noalloc_max_bytes());
        the call allocates nothing.  Calls that overlap on the GPU race: they share the array.  Outputs as bie_gmres."""
        import torch
        n = rhs.numel()
        lda = int(lda if lda is not None else A.stride(0))
        pA = _dev_f64(A, (n - 1) * lda + n)
        assert out_i32.is_cuda and out_i32.dtype == torch.int32 and out_i32.numel() >= 2
        _check(lib().bie_gmres_noalloc(self._h, n, pA, lda, _dev_f64(rhs, n), float(tol), int(restart), int(max_iters),
                                       _dev_f64(x, n), out_i32.data_ptr(), _dev_f64(out_f64, 1),
                                       out_i32.data_ptr() + 4, _stream()), "bie_gmres_noalloc")
        return x

    def bie_gmres_hybrid(self, A, ncols_dense: int, rhs, x, tol: float, restart: int, max_iters: int, workspace,
                         out_i32, out_f64, res_hist=None):
        """Asynchronous.  A: the leading ncols_dense x ncols_dense block written by bie_build_block (block format).
        Outputs as bie_gmres."""
        import torch
        n = rhs.numel()
        pA = _dev_f64(A, self.bie_hybrid_block_bytes(ncols_dense) // 8)
        assert out_i32.is_cuda and out_i32.dtype == torch.int32 and out_i32.numel() >= 2
        assert workspace.is_cuda and workspace.is_contiguous()
        ws_bytes = workspace.numel() * workspace.element_size()
        _check(lib().bie_gmres_hybrid(self._h, n, pA, int(ncols_dense), _dev_f64(rhs, n), float(tol), int(restart),
                                      int(max_iters), _dev_f64(x, n), out_i32.data_ptr(), _dev_f64(out_f64, 1),
                                      out_i32.data_ptr() + 4,
                                      None if res_hist is None else _dev_f64(res_hist, int(max_iters) + 1),
                                      workspace.data_ptr(), ws_bytes, _stream()), "bie_gmres_hybrid")
        return x

    # ---- end to end with host buffers ------------------------------------------------------------------
    @staticmethod
    def bie_solve_workspace_bytes(n: int, restart: int, matrix_free=False) -> int:
        return int(lib().bie_solve_workspace_bytes(int(n), int(restart), int(matrix_free)))

    def bie_solve_host(self, counts, kinds, zeta, dzeta, d2zeta, rhs, x, tol: float, restart: int, max_iters: int,
                       dev_workspace, matrix_free=False) -> Tuple[int, float, int]:
        """Host (ideally pinned) CPU tensors / numpy arrays in, density x (host) out; synchronises.
        -> (iters, relres_true, status)"""
        counts, kinds = _i32(counts), _i32(kinds)
        n = int(counts.sum())

        def hp(a, nbytes):
            if isinstance(a, np.ndarray):
                assert a.flags.c_contiguous and a.nbytes >= nbytes
                return a.ctypes.data
            assert (not a.is_cuda) and a.is_contiguous() and a.numel() * a.element_size() >= nbytes
            return a.data_ptr()

        iters, relres = ctypes.c_int32(), ctypes.c_double()
        ws_bytes = dev_workspace.numel() * dev_workspace.element_size()
        rc = lib().bie_solve_host(self._h, int(counts.size), _ip(counts), _ip(kinds), hp(zeta, 16 * n),
                                  hp(dzeta, 16 * n), hp(d2zeta, 16 * n), hp(rhs, 8 * n), float(tol), int(restart),
                                  int(max_iters), int(matrix_free), hp(x, 8 * n), ctypes.byref(iters),
                                  ctypes.byref(relres), dev_workspace.data_ptr(), ws_bytes, _stream())
        _check(rc, "bie_solve_host", ok=(BIE_OK, BIE_MAX_ITERS))
        return int(iters.value), float(relres.value), int(rc)

    # ---- roofline probe ----------------------------------------------------------------------------------
    def bie_probe_read(self, buf, out):
        """streams the CUDA float64 tensor `buf` once, read-only (roofline denominator of the GEMV)"""
        nbytes = (buf.numel() * buf.element_size()) // 16 * 16
        _check(lib().bie_probe_read(self._h, buf.data_ptr(), nbytes, _dev_f64(out, 1), _stream()), "bie_probe_read")

    def bie_probe_dfma(self, fma_per_thread: int, out) -> int:
        total = ctypes.c_int64()
        _check(lib().bie_probe_dfma(self._h, int(fma_per_thread), _dev_f64(out, 1), ctypes.byref(total), _stream()),
               "bie_probe_dfma")
        return int(total.value)
