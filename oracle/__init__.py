"""ctypes front-end of the CPU ORACLE (oracle/bie_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, by __graft_entry__.smoke() and by the cpu_baseline /
``--impl reference`` legs of bench.py.  Nothing under paper_2108_01786_b200/ imports this package and
this package imports nothing from it (argument marshalling below is numpy only).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bie_oracle.c")
_LIB = os.path.join(_HERE, "libbie_oracle.so")
_lib: Optional[ctypes.CDLL] = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp (no fast-math) -> oracle/libbie_oracle.so."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared",
                               "-ffp-contract=off", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        L.oracle_num_threads.restype = ctypes.c_int
        L.oracle_set_num_threads.argtypes = [ctypes.c_int]
        L.oracle_cot_half.argtypes = [ctypes.c_double, ctypes.c_double, dp, dp]
        L.oracle_build.restype = ctypes.c_int
        L.oracle_build.argtypes = [ctypes.c_int, ip, ip, dp, dp, dp, ctypes.c_int, dp, ctypes.c_long]
        L.oracle_build_rows.restype = ctypes.c_int
        L.oracle_build_rows.argtypes = [ctypes.c_int, ip, ip, dp, dp, dp, ctypes.c_int, ctypes.c_long,
                                        ctypes.POINTER(ctypes.c_long), dp]
        L.oracle_cauchy_eval.restype = ctypes.c_int
        L.oracle_cauchy_eval.argtypes = [ctypes.c_int, ip, ip, dp, dp, ctypes.c_int, dp, ctypes.c_long, dp, dp]
        L.oracle_add_cyl_columns.restype = ctypes.c_int
        L.oracle_add_cyl_columns.argtypes = [ctypes.c_int, ip, ip, dp, dp, dp, ctypes.c_long]
        L.oracle_normal_velocity_sums.restype = ctypes.c_int
        L.oracle_normal_velocity_sums.argtypes = [ctypes.c_int, ip, dp, dp, dp, dp, ctypes.c_long,
                                                  ctypes.POINTER(ctypes.c_long), dp]
        L.oracle_matvec.argtypes = [ctypes.c_long, dp, ctypes.c_long, dp, dp]
        L.oracle_matvec_rect.argtypes = [ctypes.c_long, ctypes.c_long, dp, ctypes.c_long, dp, dp]
        L.oracle_gmres.restype = ctypes.c_int
        L.oracle_gmres.argtypes = [ctypes.c_long, dp, ctypes.c_long, dp, ctypes.c_double, ctypes.c_int,
                                   ctypes.c_int, dp, ip, dp, dp]
        _lib = L
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _ip(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int))


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_num_threads(t: int) -> None:
    lib().oracle_set_num_threads(int(t))


def cot_half(x: float, y: float) -> complex:
    re = ctypes.c_double()
    im = ctypes.c_double()
    lib().oracle_cot_half(float(x), float(y), ctypes.byref(re), ctypes.byref(im))
    return complex(re.value, im.value)


def _c128_as_f64(z: np.ndarray) -> np.ndarray:
    z = np.ascontiguousarray(z, dtype=np.complex128)
    return z.view(np.float64)


def build_matrix(counts, kinds, zeta, dzeta, d2zeta, variant: int = 0,
                 out: Optional[np.ndarray] = None) -> np.ndarray:
    """Matrix of Eq. (3.16) (variant 0), the uncorrected operator B of Eq. (3.10) (variant 1), or the vortex-sheet
    system matrix of Eqs. (4.14) + (4.17) built from the adjoint matrices of Eq. (4.7) (variant 2)."""
    counts = np.ascontiguousarray(counts, dtype=np.int32)
    kinds = np.ascontiguousarray(kinds, dtype=np.int32)
    n = int(counts.sum())
    z, dz, d2z = _c128_as_f64(zeta), _c128_as_f64(dzeta), _c128_as_f64(d2zeta)
    assert z.size == 2 * n and dz.size == 2 * n and d2z.size == 2 * n
    A = out if out is not None else np.empty((n, n), dtype=np.float64)
    assert A.flags.c_contiguous and A.shape == (n, n)
    rc = lib().oracle_build(int(counts.size), _ip(counts), _ip(kinds), _dp(z), _dp(dz), _dp(d2z),
                            int(variant), _dp(A), n)
    if rc != 0:
        raise ValueError(f"oracle_build failed: {rc}")
    return A


def build_rows(counts, kinds, zeta, dzeta, d2zeta, rows, variant: int = 0) -> np.ndarray:
    """The listed rows of build_matrix's result (len(rows) x n)."""
    counts = np.ascontiguousarray(counts, dtype=np.int32)
    kinds = np.ascontiguousarray(kinds, dtype=np.int32)
    rows = np.ascontiguousarray(rows, dtype=np.int64)
    n = int(counts.sum())
    z, dz, d2z = _c128_as_f64(zeta), _c128_as_f64(dzeta), _c128_as_f64(d2zeta)
    out = np.empty((rows.size, n), dtype=np.float64)
    rc = lib().oracle_build_rows(int(counts.size), _ip(counts), _ip(kinds), _dp(z), _dp(dz), _dp(d2z),
                                 int(variant), rows.size, rows.ctypes.data_as(ctypes.POINTER(ctypes.c_long)), _dp(out))
    if rc != 0:
        raise ValueError(f"oracle_build_rows failed: {rc}")
    return out


def build_matrix_appendix_b(counts, kinds, zeta, dzeta, d2zeta, centers) -> np.ndarray:
    """Matrix of Eq. (B.2): the operator B of Eq. (3.10) plus the columns phi_cyl/psi_cyl(zeta - z_m) <1_m, .>
    (stream function prescribed on the solids; a_m = <1_m, omega> unknown).  centers: one complex z_m per obstacle."""
    A = build_matrix(counts, kinds, zeta, dzeta, d2zeta, variant=1)
    counts = np.ascontiguousarray(counts, dtype=np.int32)
    kinds = np.ascontiguousarray(kinds, dtype=np.int32)
    zc = np.ascontiguousarray(np.asarray(centers, dtype=np.complex128).reshape(-1))
    assert zc.size == int(np.sum(kinds == 2))
    zcf = zc.view(np.float64) if zc.size else np.zeros(2)
    rc = lib().oracle_add_cyl_columns(int(counts.size), _ip(counts), _ip(kinds), _dp(_c128_as_f64(zeta)), _dp(zcf), _dp(A),
                                      A.shape[1])
    if rc != 0:
        raise ValueError(f"oracle_add_cyl_columns failed: {rc}")
    return A


def cauchy_eval(counts, kinds, zeta, dzeta, fvals, zpts) -> np.ndarray:
    """Eq. (F.4) / (5.5): values at the points zpts (complex, in the closed fluid region) of nf functions analytic in the
    fluid, from their boundary values fvals (nf x n complex) -> (nf x npts complex)."""
    counts = np.ascontiguousarray(counts, dtype=np.int32)
    kinds = np.ascontiguousarray(kinds, dtype=np.int32)
    n = int(counts.sum())
    f = np.ascontiguousarray(np.atleast_2d(np.asarray(fvals, dtype=np.complex128)))
    zp = np.ascontiguousarray(np.asarray(zpts, dtype=np.complex128).reshape(-1))
    assert f.shape[1] == n
    out = np.empty((f.shape[0], zp.size), dtype=np.complex128)
    rc = lib().oracle_cauchy_eval(int(counts.size), _ip(counts), _ip(kinds), _dp(_c128_as_f64(zeta)), _dp(_c128_as_f64(dzeta)),
                                  int(f.shape[0]), _dp(f.view(np.float64)), zp.size, _dp(zp.view(np.float64)),
                                  _dp(out.view(np.float64)))
    if rc != 0:
        raise ValueError(f"oracle_cauchy_eval failed: {rc}")
    return out


def hilbert(f: np.ndarray) -> np.ndarray:
    """Periodic Hilbert transform of Eq. (3.22) on equispaced samples, by the FFT with the symbol
    -i sgn(k); the Nyquist mode of an even-length sample has no sign and is dropped."""
    f = np.asarray(f, dtype=np.float64)
    M = f.size
    k = np.fft.fftfreq(M, d=1.0 / M)
    sym = -1j * np.sign(k)
    if M % 2 == 0:
        sym[M // 2] = 0.0
    return np.real(np.fft.ifft(sym * np.fft.fft(f)))


def normal_velocity(counts, zeta, dzeta, d2zeta, domega, rows=None) -> np.ndarray:
    """s_alpha * dphi~/dn on Gamma_0 at the listed nodes (default: all) from the derivatives omega' of the densities:
    the sum of Eq. (3.19) over the solids and Eq. (3.24),
        -1/2 H omega'_0  -  G+_00 omega'_0  +  sum_j K+_j0 omega'_j,
    WITHOUT the phi_mv term (3.17).  Hilbert transform by FFT, the integrals by the trapezoidal rule."""
    counts = np.ascontiguousarray(counts, dtype=np.int32)
    n, M0 = int(counts.sum()), int(counts[0])
    z, dz, d2z = _c128_as_f64(zeta), _c128_as_f64(dzeta), _c128_as_f64(d2zeta)
    w = np.ascontiguousarray(domega, dtype=np.float64)
    assert w.size == n
    rows = np.arange(M0, dtype=np.int64) if rows is None else np.ascontiguousarray(rows, dtype=np.int64)
    out = np.empty(rows.size, dtype=np.float64)
    rc = lib().oracle_normal_velocity_sums(int(counts.size), _ip(counts), _dp(z), _dp(dz), _dp(d2z), _dp(w), rows.size,
                                           rows.ctypes.data_as(ctypes.POINTER(ctypes.c_long)), _dp(out))
    if rc != 0:
        raise ValueError(f"oracle_normal_velocity_sums failed: {rc}")
    return out - 0.5 * hilbert(w[:M0])[rows]


def matvec(A: np.ndarray, x: np.ndarray, lda: Optional[int] = None) -> np.ndarray:
    """y = A x for a C-contiguous (nrows x ncols) block, ncols = len(x).  With ``lda`` given, A is the flat (or 2-D)
    storage of a row-major matrix whose rows are lda doubles apart and only the first len(x) columns of each are used."""
    A = np.ascontiguousarray(A, dtype=np.float64)
    x = np.ascontiguousarray(x, dtype=np.float64)
    if lda is None:
        nrows, ncols = A.shape
        lda = ncols
    else:
        ncols = x.size
        assert lda >= ncols and A.size % lda == 0
        nrows = A.size // lda
    assert x.size == ncols
    y = np.empty(nrows, dtype=np.float64)
    lib().oracle_matvec_rect(nrows, ncols, _dp(A), int(lda), _dp(x), _dp(y))
    return y


def gmres(A: np.ndarray, b: np.ndarray, tol: float = 1e-13, restart: int = 50,
          max_iters: int = 1000) -> Tuple[np.ndarray, int, float, np.ndarray, int]:
    """-> (x, iters, relres_true, res_hist[0..iters], status)   status 0 = converged, 1 = max_iters."""
    A = np.ascontiguousarray(A, dtype=np.float64)
    b = np.ascontiguousarray(b, dtype=np.float64)
    n = A.shape[0]
    x = np.empty(n, dtype=np.float64)
    hist = np.zeros(max_iters + 1, dtype=np.float64)
    iters = ctypes.c_int()
    relres = ctypes.c_double()
    rc = lib().oracle_gmres(n, _dp(A), A.shape[1], _dp(b), float(tol), int(restart), int(max_iters),
                            _dp(x), ctypes.byref(iters), ctypes.byref(relres), _dp(hist))
    if rc < 0:
        raise ValueError(f"oracle_gmres failed: {rc}")
    return x, int(iters.value), float(relres.value), hist[:iters.value + 1].copy(), int(rc)
