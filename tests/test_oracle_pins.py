"""Pins of the CPU oracle (oracle/) against what the paper and the mathematics fix.  CPU only.

Each test names the passage it pins (PAPER.md = /root/reference/PAPER.md) and the mistake it is
meant to catch.  None of them re-types the oracle's own formula: they use 40-digit values (mpmath,
stored under tests/golden/), closed forms, invariants from Eq. (6.3), adaptive quadrature of the
kernels of Table 1 written with numpy's complex tan (not the oracle's half-angle form), the
Cauchy-integral reproduction of an analytic function, and LAPACK.
"""
import os

import numpy as np
import pytest

import oracle
from paper_2108_01786_b200 import inputs

HERE = os.path.dirname(os.path.abspath(__file__))


def _build(geo, variant=0):
    return oracle.build_matrix(geo.counts, geo.kinds, geo.zeta, geo.dzeta, geo.d2zeta, variant)


# --------------------------------------------------------------------------------------------
# P1  the per-pair arithmetic: cot((x+iy)/2), Eq. (3.4)
# --------------------------------------------------------------------------------------------
def _golden_cot():
    rows = []
    with open(os.path.join(HERE, "golden", "cot_half_40digits.txt")) as f:
        for line in f:
            if line.startswith("#"):
                continue
            xh, yh, re, im = line.split()
            rows.append((float.fromhex(xh), float.fromhex(yh), float(re), float(im)))
    return rows


def test_p1_cot_against_40_digit_values():
    """A wrong sign, a missing half angle or a cancellation-prone denominator fails here."""
    worst = 0.0
    for x, y, re, im in _golden_cot():
        c = oracle.cot_half(x, y)
        ref = complex(re, im)
        # the argument x is reduced mod 2 pi inside sin/cos: allow eps*|x|/dist-to-pole conditioning
        w = complex(x, y)
        dist = min(abs(w - 2 * np.pi * k) for k in range(-3, 4))
        cond = 1.0 + abs(x) / max(dist, 1e-300)
        err = abs(c - ref) / abs(ref)
        assert err <= 4e-16 * cond + 4e-16, (x, y, err)
        worst = max(worst, err)
    assert worst < 1e-9


def test_p1_cot_is_the_periodic_image_sum():
    """Eq. (3.4): (1/2)cot(w/2) = PV sum_k 1/(w + 2 pi k); symmetric truncation error is O(1/K)."""
    rng = np.random.default_rng(1)
    K = 200000
    k = np.arange(1, K + 1, dtype=np.float64)
    for _ in range(5):
        w = complex(rng.uniform(-3, 3), rng.uniform(-2, 2))
        s = 1.0 / w + np.sum(1.0 / (w + 2 * np.pi * k) + 1.0 / (w - 2 * np.pi * k))
        c = 0.5 * oracle.cot_half(w.real, w.imag)
        assert abs(s - c) < 5.0 * abs(w) / K + 1e-9


def test_p1_flat_over_flat_entry_closed_form():
    """zeta_0 = a, zeta_1 = a - iH: G_01 = (1/2) sin x/(cosh H - cos x), K_00 = K_11 = 0
    (follows from Table 1, with zeta' = 1)."""
    M0, M1, H = 24, 20, 0.7
    geo = inputs.flat_flat(M0, M1, H)
    B = _build(geo, variant=1)
    a0 = 2 * np.pi * np.arange(M0) / M0
    a1 = 2 * np.pi * np.arange(M1) / M1
    x = a1[None, :] - a0[:, None]
    G01 = 0.5 * np.sin(x) / (np.cosh(H) - np.cos(x)) / M1
    assert np.max(np.abs(B[:M0, M0:] - G01)) < 1e-15
    # -G_10: source on the surface, target on the bottom: w = a0 - a1 + iH
    x = a0[None, :] - a1[:, None]
    G10 = 0.5 * np.sin(x) / (np.cosh(H) - np.cos(x)) / M0
    assert np.max(np.abs(B[M0:, :M0] + G10)) < 1e-15
    assert np.max(np.abs(B[:M0, :M0] + 0.5 * np.eye(M0))) < 1e-16
    assert np.max(np.abs(B[M0:, M0:] - 0.5 * np.eye(M1))) < 1e-16


# --------------------------------------------------------------------------------------------
# P2  block row sums from Eq. (6.3)
# --------------------------------------------------------------------------------------------
def test_p2_block_row_sums_config1():
    """Constant densities: Phi_0 = -+omega_0/2 above/below Gamma_0, Phi_1 = +-i omega_1/2, Phi_j = 0
    outside / -i omega_j inside obstacle j.  Pins the +-1/2, orientation, Re/Im selection, the
    diagonal term, the weights 1/M_j and E_m."""
    P = inputs.make_config(1)
    g = P.geometry
    B = _build(g, variant=1)
    A = _build(g, variant=0)
    s0, s1, s2 = g.component(0), g.component(1), g.component(2)
    one = lambda s: np.where((np.arange(g.n) >= s.start) & (np.arange(g.n) < s.stop), 1.0, 0.0)
    tol = 2e-14
    r = B @ one(s0)  # omega = 1_0: phi~ on Gamma_0^- is -1/2; psi~ on solids is 0
    assert np.max(np.abs(r[s0] + 0.5)) < tol and np.max(np.abs(r[s1.start:])) < tol
    r = B @ one(s1)  # omega = 1_1: Phi_1 = i/2 above the bottom: phi~ = 0 on Gamma_0, psi~ = 1/2 on solids
    assert np.max(np.abs(r[s0])) < tol and np.max(np.abs(r[s1.start:] - 0.5)) < tol
    r = B @ one(s2)  # kernel of B (3.12)
    assert np.max(np.abs(r)) < tol
    r = A @ one(s2)  # A 1_m = -1_m  (3.13)
    assert np.max(np.abs(r + one(s2))) < tol
    # block-wise statements
    assert np.max(np.abs(B[s0, s0].sum(1) + 0.5)) < tol        # K_00 1 = 0
    assert np.max(np.abs(B[s2, s2].sum(1))) < tol              # (1/2 I + K_22) 1 = 0  => K_22 1 = -1/2
    assert np.max(np.abs(B[s2, s1].sum(1) - 0.5)) < tol        # K_21 1 = 1/2
    assert np.max(np.abs(B[s1, s2].sum(1))) < tol              # K_12 1 = 0
    assert np.max(np.abs(B[s1, s0].sum(1))) < tol              # G_10 1 = 0
    assert np.max(np.abs(B[s0, s2].sum(1))) < tol              # G_02 1 = 0
    # E_m only touches the obstacle's diagonal block
    D = A - B
    mask = np.zeros_like(D, dtype=bool)
    mask[s2, s2] = True
    assert np.max(np.abs(D[~mask])) == 0.0
    assert np.max(np.abs(D[s2, s2] + 1.0 / g.counts[2])) < 1e-17


def test_p2_row_sums_ragged_two_obstacles():
    P = inputs.small_problem(96, 80, [48, 40], seed=3)
    g = P.geometry
    B = _build(g, variant=1)
    A = _build(g, variant=0)
    for m in (2, 3):
        v = np.zeros(g.n)
        v[g.component(m)] = 1.0
        assert np.max(np.abs(B @ v)) < 1e-12
        assert np.max(np.abs(A @ v + v)) < 1e-12


def test_counterclockwise_obstacle_breaks_the_kernel():
    """Orientation is part of the contract (reading R1): with a counter-clockwise
    ellipse (1/2 I + K_mm) 1 = 1 instead of 0."""
    P = inputs.make_config(1)
    g = P.geometry
    s2 = g.component(2)
    # reverse the parameterisation of the obstacle: a -> -a
    idx = np.r_[0, np.arange(g.counts[2] - 1, 0, -1)] + s2.start
    z, dz, d2z = g.zeta.copy(), g.dzeta.copy(), g.d2zeta.copy()
    z[s2], dz[s2], d2z[s2] = g.zeta[idx], -g.dzeta[idx], g.d2zeta[idx]
    B = oracle.build_matrix(g.counts, g.kinds, z, dz, d2z, 1)
    assert np.max(np.abs(B[s2, s2].sum(1) - 1.0)) < 1e-13


# --------------------------------------------------------------------------------------------
# P3 / P4  Cauchy-integral reproduction of an analytic function (north_star check)
# --------------------------------------------------------------------------------------------
def _cauchy_sum(g, omega, zpts):
    """Trapezoid rule for Eq. (3.3), written with numpy's complex tan:
    Phi_0(z) = (1/2 pi i) int (1/2)cot((zeta_0 - z)/2) omega_0 zeta_0' da, solids carry an extra i."""
    out = np.zeros(len(zpts), dtype=np.complex128)
    for k in range(g.counts.size):
        s = g.component(k)
        sig = 1.0 if g.kinds[k] == inputs.KIND_SURFACE else 1j
        Mk = int(g.counts[k])
        for i, z in enumerate(zpts):
            ker = 0.5 / np.tan(0.5 * (g.zeta[s] - z))
            out[i] += (sig / (1j * Mk)) * np.sum(ker * omega[s] * g.dzeta[s])
    return out


def _interior_points():
    return np.array([0.3 - 0.4j, 2.0 - 0.5j, 4.0 - 1.5j, 5.5 - 0.45j, 1.0 - 1.6j, 3.1 - 0.3j])


def _f_poles(z):
    """2 pi-periodic, analytic in the fluid of the config-1-like geometries, with poles above the free
    surface, inside the obstacle and below the bottom, so that ALL densities are excited (the entire
    function e^{iz} alone is reproduced by the bottom density only: omega_0 = omega_2 = 0)."""
    cot = lambda w: 1.0 / np.tan(w)
    return (np.exp(1j * z) + 0.3 * cot(0.5 * (z - (1.0 + 0.6j)))
            + (0.1 + 0.04j) * cot(0.5 * (z - (-1.0j))) + 0.1j * cot(0.5 * (z - (2.0 - 2.6j))))


def _reproduction_error(g, f=_f_poles):
    b = inputs.rhs_analytic(g, f)
    A = _build(g)
    x, iters, relres, hist, status = oracle.gmres(A, b, 1e-14, 60, 400)
    assert status == 0
    zp = _interior_points()
    return np.max(np.abs(_cauchy_sum(g, x, zp) - f(zp))), x


def test_p3_entire_function_uses_the_bottom_density_only():
    """f = e^{iz} (config 1's right-hand side) is entire and decays upwards: no jump across Gamma_0 or the
    obstacle, so omega_0 = 0 and omega_2 = 0 and Phi_1 alone reproduces f."""
    P = inputs.make_config(1)
    g = P.geometry
    err, x = _reproduction_error(g, lambda z: np.exp(1j * z))
    assert err < 2e-14
    assert np.max(np.abs(x[g.component(0)])) < 1e-13 and np.max(np.abs(x[g.component(2)])) < 1e-13
    assert np.max(np.abs(x[g.component(1)])) > 1.0


def test_p3_analytic_function_reproduction_config1():
    """b_0 = Re f, b_k = Im f for f = e^{iz}; by the uniqueness argument the sum of
    Cauchy integrals equals f inside the fluid and <1_m, omega> = 0.  End-to-end pin of the whole
    matrix (Plemelj 1/2, signs, Re/Im pattern, weights, diagonal, E_m) and of the solver."""
    P = inputs.make_config(1)
    g = P.geometry
    err, x = _reproduction_error(g)
    assert err < 2e-13, err
    assert abs(np.mean(x[g.component(2)])) < 1e-13          # psi|_2 = <1_2, omega> = 0
    for k in range(3):                                      # every density is excited by this f
        assert np.max(np.abs(x[g.component(k)])) > 0.05


def test_p3_fails_without_the_pieces():
    """Mutation check of the pin itself: dropping the diagonal limit, flipping the sign of the
    -G_k0 blocks, or using weights 1/M_k (target) instead of 1/M_j (source) must break P3."""
    P = inputs.make_config(1)
    g = P.geometry
    f = _f_poles
    b = inputs.rhs_analytic(g, f)
    A = _build(g)
    zp = _interior_points()
    s0 = g.component(0)

    def err_of(Am):
        x = np.linalg.solve(Am, b)
        return np.max(np.abs(_cauchy_sum(g, x, zp) - f(zp)))

    assert err_of(A) < 2e-13
    A1 = A.copy()
    d = np.arange(g.n)
    diag_k = np.imag(g.d2zeta / (2 * g.dzeta)) / np.repeat(g.counts, g.counts)
    A1[d, d] -= diag_k
    assert err_of(A1) > 1e-6
    A2 = A.copy()
    A2[s0.stop:, s0] *= -1.0
    assert err_of(A2) > 1e-3
    A3 = A.copy()
    A3[s0, s0.stop:] *= -1.0
    assert err_of(A3) > 1e-3


def test_p4_spectral_convergence():
    """Trapezoid collocation is spectrally accurate: the reproduction error decays
    geometrically under refinement M -> 2M until roundoff."""
    errs = []
    for M in (16, 32, 64, 128, 256):
        eta = inputs.Series(np.array([1.0, 2.0]), np.array([0.05 + 0j, 0.01 - 0.02j]))
        geo = inputs.assemble([inputs.graph_curve(M, 0.0, eta),
                               inputs.graph_curve(M, -2.0, None),
                               inputs.ellipse_curve(M, -1.0j, 0.4, 0.2, 0.3)], [0, 1, 2])
        errs.append(_reproduction_error(geo)[0])
    assert errs[0] > 1e-3                    # under-resolved: the pin is sensitive
    assert errs[1] < errs[0] / 10
    assert errs[2] < errs[1] / 100
    assert errs[3] < errs[2] / 1e4           # error ~ e^{-c M}: the decrements grow
    assert errs[4] < 5e-14, errs             # roundoff floor


# --------------------------------------------------------------------------------------------
# P5  adaptive quadrature of the kernels of Table 1 on tiny inputs
# --------------------------------------------------------------------------------------------
def test_p5_rows_against_adaptive_quadrature():
    """(1/2pi) int K_kj(alpha_m, beta) omega(beta) d beta by Gauss-Kronrod (scipy quad) on analytic
    curves, integrand written from Table 1 with numpy's tan and set to the limit
    Im{zeta''/(2 zeta')} at beta = alpha; compared with (matrix row) . (samples).
    A missing diagonal term leaves an O(1/M) error; a wrong Re/Im or sign is O(1)."""
    from scipy.integrate import quad

    M0, M1, M2 = 64, 48, 40
    c0 = lambda a: a + 1j * (0.1 * np.cos(a) + 0.03 * np.sin(2 * a))
    d0 = lambda a: 1 + 1j * (-0.1 * np.sin(a) + 0.06 * np.cos(2 * a))
    e0 = lambda a: 1j * (-0.1 * np.cos(a) - 0.12 * np.sin(2 * a))
    c1 = lambda a: a + 1j * (-1.5 + 0.2 * np.cos(a))
    d1 = lambda a: 1 + 1j * (-0.2 * np.sin(a))
    e1 = lambda a: 1j * (-0.2 * np.cos(a))
    rot, zc, q, bb = np.exp(0.4j), 3.0 - 0.7j, 0.35, 0.2
    c2 = lambda a: zc + rot * (q * np.cos(a) - 1j * bb * np.sin(a))
    d2 = lambda a: rot * (-q * np.sin(a) - 1j * bb * np.cos(a))
    e2 = lambda a: rot * (-q * np.cos(a) + 1j * bb * np.sin(a))
    curves = [(c0, d0, e0, M0), (c1, d1, e1, M1), (c2, d2, e2, M2)]
    parts = []
    for c, d, e, M in curves:
        a = 2 * np.pi * np.arange(M) / M
        parts.append((c(a), d(a), e(a)))
    geo = inputs.assemble(parts, [0, 1, 2])
    B = _build(geo, variant=1)
    om = lambda b: 1.0 + 0.5 * np.cos(b) + 0.25 * np.sin(2 * b)

    def kern(k, j, a, b):
        ck, cj, dj, ej = curves[k][0], curves[j][0], curves[j][1], curves[j][2]
        if k == j and abs(b - a) < 1e-9:
            c = ej(a) / (2 * dj(a))
        else:
            c = 0.5 * dj(b) / np.tan(0.5 * (cj(b) - ck(a)))
        if k == 0 and j == 0:
            return c.imag
        if k == 0:
            return c.real
        if j == 0:
            return -c.real
        return c.imag

    for (k, m) in [(0, 5), (1, 17), (2, 3), (2, 21), (0, 40)]:
        a = 2 * np.pi * m / curves[k][3]
        row = geo.component(k).start + m
        for j in range(3):
            val, _ = quad(lambda b: kern(k, j, a, b) * om(b) / (2 * np.pi), 0, 2 * np.pi,
                          points=[a] if k == j and a > 0 else None, epsabs=1e-13, epsrel=1e-13, limit=400)
            sj = geo.component(j)
            bj = 2 * np.pi * np.arange(curves[j][3]) / curves[j][3]
            num = B[row, sj] @ om(bj)
            if k == j:  # remove the +-1/2 identity
                num -= (-0.5 if k == 0 else 0.5) * om(a)
            assert abs(num - val) < 2e-11, (k, m, j, num, val)


# --------------------------------------------------------------------------------------------
# P6  flat surface over flat bottom: closed-form solution of the linear system
# --------------------------------------------------------------------------------------------
def test_p6_flat_flat_closed_form_solution():
    """zeta_0 = a, zeta_1 = a - iH, b = (cos p a, 0):  omega_0 = -2 cos(pa)/(1+e^{-2pH}),
    omega_1 = 2 e^{-pH} sin(pa)/(1+e^{-2pH})  (Fourier analysis of Table 1 for flat boundaries)."""
    M0, M1, H, p = 64, 48, 1.3, 3
    geo = inputs.flat_flat(M0, M1, H)
    A = _build(geo)
    a0 = 2 * np.pi * np.arange(M0) / M0
    a1 = 2 * np.pi * np.arange(M1) / M1
    # operator identities G_01 cos(p.) = -1/2 e^{-pH} sin(p.), G_01 sin(p.) = 1/2 e^{-pH} cos(p.)
    G01 = A[:M0, M0:]
    assert np.max(np.abs(G01 @ np.cos(p * a1) + 0.5 * np.exp(-p * H) * np.sin(p * a0))) < 1e-14
    assert np.max(np.abs(G01 @ np.sin(p * a1) - 0.5 * np.exp(-p * H) * np.cos(p * a0))) < 1e-14
    b = np.concatenate([np.cos(p * a0), np.zeros(M1)])
    x, iters, relres, hist, status = oracle.gmres(A, b, 1e-14, 50, 200)
    assert status == 0 and relres < 1e-13
    den = 1 + np.exp(-2 * p * H)
    assert np.max(np.abs(x[:M0] + 2 * np.cos(p * a0) / den)) < 1e-13
    assert np.max(np.abs(x[M0:] - 2 * np.exp(-p * H) * np.sin(p * a1) / den)) < 1e-13


# --------------------------------------------------------------------------------------------
# P7  GMRES against LAPACK and its own invariants
# --------------------------------------------------------------------------------------------
def test_p7_gmres_matches_lapack_and_is_monotone():
    rng = np.random.default_rng(11)
    n = 120
    A = np.eye(n) * 0.5 + rng.standard_normal((n, n)) / (4 * np.sqrt(n))
    b = rng.standard_normal(n)
    xref = np.linalg.solve(A, b)
    for restart in (n, 25, 7):
        x, iters, relres, hist, status = oracle.gmres(A, b, 1e-13, restart, 2000)
        assert status == 0
        assert relres <= 2e-13
        assert np.linalg.norm(x - xref) / np.linalg.norm(xref) < 1e-11
        assert np.all(np.diff(hist) <= 1e-15), "recurrence residual must not increase"
        assert hist[-1] <= 1e-13 and (iters < 2 or hist[-2] > 1e-13), "stops at the first step below tol"
        assert iters <= n if restart == n else True
    # unrestarted GMRES terminates in at most n steps on any nonsingular matrix
    x, iters, *_ = oracle.gmres(A, b, 1e-13, n, 2000)
    assert iters <= n


def test_p7_gmres_krylov_exactness_low_rank():
    """A = I + (rank-3): GMRES converges in at most 4 steps (minimal polynomial degree 4)."""
    rng = np.random.default_rng(2)
    n = 60
    U = rng.standard_normal((n, 3))
    W = rng.standard_normal((n, 3))
    A = np.eye(n) + U @ W.T / n
    b = rng.standard_normal(n)
    x, iters, relres, hist, status = oracle.gmres(A, b, 1e-12, 30, 100)
    assert status == 0 and iters <= 4
    assert np.linalg.norm(A @ x - b) / np.linalg.norm(b) < 1e-12


def test_p7_gmres_edge_cases():
    A = np.array([[2.0, 0.0], [0.0, 4.0]])
    x, iters, relres, hist, status = oracle.gmres(A, np.zeros(2), 1e-13, 5, 10)
    assert iters == 0 and status == 0 and np.all(x == 0)
    x, iters, relres, hist, status = oracle.gmres(A, np.array([1.0, 1.0]), 1e-13, 5, 1)
    assert iters == 1 and status == 1  # max_iters reached, x is the 1-step minimiser
    x, iters, relres, hist, status = oracle.gmres(A, np.array([1.0, 0.0]), 1e-13, 5, 10)
    assert iters == 1 and status == 0 and abs(x[0] - 0.5) < 1e-16  # lucky breakdown


def test_matvec_is_the_plain_definition():
    import math
    rng = np.random.default_rng(4)
    A = rng.standard_normal((37, 37))
    x = rng.standard_normal(37)
    y = oracle.matvec(A, x)
    for i in (0, 13, 36):
        assert abs(y[i] - math.fsum(A[i, j] * x[j] for j in range(37))) < 1e-14
    # rectangular blocks (nrows != ncols, both ways) and a leading dimension larger than the column count: an index slip
    # (i * ncols instead of i * lda, rows and columns swapped, a column of the padding read) fails one of these
    for nrows, ncols, lda in ((5, 41, 41), (41, 5, 5), (7, 13, 20), (23, 9, 9 + 3), (1, 6, 8)):
        S = rng.standard_normal((nrows, lda))
        S[:, ncols:] = 1.0e6                     # padding columns must never be read
        x = rng.standard_normal(ncols)
        y = oracle.matvec(np.ascontiguousarray(S[:, :ncols]), x) if lda == ncols else oracle.matvec(S, x, lda=lda)
        assert y.shape == (nrows,)
        for i in range(nrows):
            assert abs(y[i] - math.fsum(S[i, j] * x[j] for j in range(ncols))) < 1e-13, (nrows, ncols, lda, i)


@pytest.mark.parametrize("variant", [0, 1, 2])
def test_build_rows_is_rows_of_build_matrix(variant):
    """oracle.build_rows (what the full-size GPU parity tests compare against) is, bit for bit, the listed rows of
    oracle.build_matrix (what pins P1-P8 fix) -- for unsorted, repeated and boundary rows, with and without an obstacle"""
    rng = np.random.default_rng(variant)
    for g in (inputs.make_config(1).geometry, inputs.small_problem(37, 29, [19, 23], seed=3).geometry,
              inputs.small_problem(5, 3, [], seed=1).geometry):
        A = _build(g, variant)
        n = g.n
        off = g.offsets
        rows = list(rng.integers(0, n, size=min(n, 25)))
        rows += [n - 1, 0, 0, n - 1] + [int(o) for o in off[:-1]] + [int(o) - 1 for o in off[1:]]
        rows = np.array(rows, dtype=np.int64)
        rng.shuffle(rows)
        R = oracle.build_rows(g.counts, g.kinds, g.zeta, g.dzeta, g.d2zeta, rows, variant=variant)
        assert R.shape == (rows.size, n)
        assert np.array_equal(R, A[rows])
        # one row at a time and in reverse order give the same bits
        R1 = oracle.build_rows(g.counts, g.kinds, g.zeta, g.dzeta, g.d2zeta, rows[::-1], variant=variant)
        assert np.array_equal(R1, A[rows[::-1]])
        assert np.array_equal(oracle.build_rows(g.counts, g.kinds, g.zeta, g.dzeta, g.d2zeta, rows[:1], variant=variant)[0],
                              A[rows[0]])
    with pytest.raises(ValueError):
        oracle.build_rows(g.counts, g.kinds, g.zeta, g.dzeta, g.d2zeta, np.array([g.n]), variant=variant)


def test_config_iteration_counts_in_paper_range():
    """Plausibility only (i_max 30-120 at tol 1e-15): configs 1-2 at tol 1e-13."""
    for c, lo, hi in ((1, 10, 40), (2, 20, 60)):
        P = inputs.make_config(c)
        A = _build(P.geometry)
        x, iters, relres, hist, status = oracle.gmres(A, P.rhs[0], P.tol, P.restart, P.max_iters)
        assert status == 0 and lo <= iters <= hi and relres < 2e-13


# --------------------------------------------------------------------------------------------
# P8  vortex-sheet system (variant 2): adjoint matrices of Eq. (4.7), systems (4.5) and (4.14) + (4.17)
# --------------------------------------------------------------------------------------------
def _comp_of(geo):
    return np.repeat(np.arange(len(geo.counts)), geo.counts)


@pytest.mark.parametrize("which", ["config1", "ragged"])
def test_p8_dagger_relation_against_the_pinned_B(which):
    """Eq. (4.7): (K+_jk)_ml = (M_k/M_j) K_jk,lm, same for G+.  Hence the matrix S of (4.14) + (4.17),
    which the oracle builds entry by entry from K_jk(alpha_jl, alpha_km)/M_j, must equal D B^T D^-1 + J with B the
    operator of Eq. (3.10) (pinned by P1-P6), D = diag(M of the node's component) and J = +1 on Gamma_0 rows
    (1/2 I + K+_00 against (-1/2 I + K_00)^T), -1 on solid rows.  A wrong weight (1/M_k for 1/M_j), a wrong sign of the
    cot argument, a swapped Re/Im or a zeta' taken from the column node each break it at O(1)."""
    geo = inputs.make_config(1).geometry if which == "config1" else inputs.small_problem(37, 29, [19, 23]).geometry
    B = _build(geo, variant=1)
    S = _build(geo, variant=2)
    comp = _comp_of(geo)
    D = np.asarray(geo.counts, dtype=float)[comp]
    J = np.where(comp == 0, 1.0, -1.0)
    R = D[:, None] * B.T / D[None, :] + np.diag(J)
    assert np.max(np.abs(S - R)) < 5e-15
    # and it is NOT the plain transpose when the components have different M (the re-normalisation matters)
    assert np.max(np.abs(S - (B.T + np.diag(J)))) > 1e-3


def test_p8_flat_bottom_auxiliary_system_closed_form():
    """N = 1, flat surface zeta_0 = a over a flat bottom zeta_1 = a - iH: K+_11 = 0, so Eq. (4.5) is
    -1/2 gamma_1 = -G+_01 gamma_0.  From cot(z/2) = i (1 + 2 sum_k e^{-ikz}) for Im z < 0:
    G_01(beta, alpha) = Re{1/2 cot((alpha - beta - iH)/2)} = sum_k e^{-kH} sin k(alpha - beta), hence
    G+_01 cos(p.) = 1/2 e^{-pH} sin(p.), G+_01 sin(p.) = -1/2 e^{-pH} cos(p.), and gamma_1 = e^{-pH} sin(p a) for
    gamma_0 = cos(p a).  Also K+_00 = 0 and G+_10 = the mirror image (row on Gamma_0 lies ABOVE the source)."""
    M0, M1, H, p = 64, 48, 1.3, 3
    geo = inputs.flat_flat(M0, M1, H)
    S = _build(geo, variant=2)
    a0 = 2 * np.pi * np.arange(M0) / M0
    a1 = 2 * np.pi * np.arange(M1) / M1
    G01 = S[M0:, :M0]                     # rows on the bottom, columns on Gamma_0
    assert np.max(np.abs(G01 @ np.cos(p * a0) - 0.5 * np.exp(-p * H) * np.sin(p * a1))) < 1e-14
    assert np.max(np.abs(G01 @ np.sin(p * a0) + 0.5 * np.exp(-p * H) * np.cos(p * a1))) < 1e-14
    assert np.max(np.abs(S[:M0, :M0] - 0.5 * np.eye(M0))) < 1e-15      # 1/2 I + K+_00, K+_00 = 0
    assert np.max(np.abs(S[M0:, M0:] + 0.5 * np.eye(M1))) < 1e-15      # -1/2 I + K+_11, K+_11 = 0
    # -G+_10: the bottom seen from above, Im z > 0: cot(z/2) = -i (1 + 2 sum e^{ikz}), Re{1/2 cot((a - b + iH)/2)} =
    # sum_k e^{-kH} sin k(a - b) again, so G+_10 cos(p.) = 1/2 e^{-pH} sin(p.) and the block -G+_10 gives minus that
    mG10 = S[:M0, M0:]
    assert np.max(np.abs(mG10 @ np.cos(p * a1) + 0.5 * np.exp(-p * H) * np.sin(p * a0))) < 1e-14
    # the auxiliary system (4.5), solved by the oracle's GMRES
    aux = S[M0:, M0:]
    rhs = -G01 @ np.cos(p * a0)
    x, iters, relres, hist, status = oracle.gmres(np.ascontiguousarray(aux), rhs, 1e-14, 50, 200)
    assert status == 0 and np.max(np.abs(x - np.exp(-p * H) * np.sin(p * a1))) < 1e-13


def test_p8_adjoint_rows_against_adaptive_quadrature():
    """Eq. (4.6): (K*_jk gamma_j)(alpha) = (1/2pi) int K_jk(beta, alpha) gamma_j(beta) d beta and the same
    with G, by Gauss-Kronrod on analytic curves; K_jk(beta, alpha) = Im{zeta'_k(alpha)/2 cot((zeta_k(alpha) - zeta_j(beta))/2)}
    written from Table 1 with numpy's tan, limit Im{zeta''/(2 zeta')} at beta = alpha; against (row of S) . samples."""
    from scipy.integrate import quad

    M0, M1, M2 = 64, 48, 40
    c0 = lambda a: a + 1j * (0.1 * np.cos(a) + 0.03 * np.sin(2 * a))
    d0 = lambda a: 1 + 1j * (-0.1 * np.sin(a) + 0.06 * np.cos(2 * a))
    e0 = lambda a: 1j * (-0.1 * np.cos(a) - 0.12 * np.sin(2 * a))
    c1 = lambda a: a + 1j * (-1.5 + 0.2 * np.cos(a))
    d1 = lambda a: 1 + 1j * (-0.2 * np.sin(a))
    e1 = lambda a: 1j * (-0.2 * np.cos(a))
    rot, zc, q, bb = np.exp(0.4j), 3.0 - 0.7j, 0.35, 0.2
    c2 = lambda a: zc + rot * (q * np.cos(a) - 1j * bb * np.sin(a))
    d2 = lambda a: rot * (-q * np.sin(a) - 1j * bb * np.cos(a))
    e2 = lambda a: rot * (-q * np.cos(a) + 1j * bb * np.sin(a))
    curves = [(c0, d0, e0, M0), (c1, d1, e1, M1), (c2, d2, e2, M2)]
    parts = []
    for c, d, e, M in curves:
        a = 2 * np.pi * np.arange(M) / M
        parts.append((c(a), d(a), e(a)))
    geo = inputs.assemble(parts, [0, 1, 2])
    S = _build(geo, variant=2)
    gam = lambda b: 0.7 + 0.5 * np.cos(b) - 0.25 * np.sin(3 * b)

    def kern(k, j, a, b):
        """entry pattern of row block k (point alpha on Gamma_k), column block j (density on Gamma_j)"""
        ck, dk, ek, cj = curves[k][0], curves[k][1], curves[k][2], curves[j][0]
        if k == j and abs(b - a) < 1e-9:
            c = ek(a) / (2 * dk(a))
        else:
            c = 0.5 * dk(a) / np.tan(0.5 * (ck(a) - cj(b)))
        if k == 0 and j == 0:
            return c.imag          # K*_00   (Eq. 4.14)
        if k == 0:
            return -c.real         # -G*_j0  (Eq. 4.14)
        if j == 0:
            return c.real          # G*_0k   (Eq. 4.17)
        return c.imag              # K*_jk   (Eq. 4.5 / 4.17)

    for (k, m) in [(0, 5), (1, 17), (2, 3), (2, 21), (0, 40)]:
        a = 2 * np.pi * m / curves[k][3]
        row = geo.component(k).start + m
        for j in range(3):
            val, _ = quad(lambda b: kern(k, j, a, b) * gam(b) / (2 * np.pi), 0, 2 * np.pi,
                          points=[a] if k == j and a > 0 else None, epsabs=1e-13, epsrel=1e-13, limit=400)
            sj = geo.component(j)
            bj = 2 * np.pi * np.arange(curves[j][3]) / curves[j][3]
            num = S[row, sj] @ gam(bj)
            if k == j:  # remove the +-1/2 identity
                num -= (0.5 if k == 0 else -0.5) * gam(a)
            assert abs(num - val) < 2e-11, (k, m, j, num, val)


def test_p8_auxiliary_system_is_well_conditioned_and_converges_like_the_paper():
    """Eq. (4.5) "is well-conditioned once enough grid points are used"; the paper's GMRES needs 20-32
    iterations on it.  Plausibility band only."""
    P = inputs.make_config(2)
    g = P.geometry
    S = _build(g, variant=2)
    M0 = g.counts[0]
    aux = np.ascontiguousarray(S[M0:, M0:])
    assert np.linalg.cond(aux) < 50
    rhs = np.cos(np.arange(aux.shape[0]) * 0.01) + 0.3
    x, iters, relres, hist, status = oracle.gmres(aux, rhs, 1e-13, 50, 500)
    assert status == 0 and 8 <= iters <= 60 and relres < 1e-12


# --------------------------------------------------------------------------------------------
# P9  normal velocity on the free surface (NEXT-2): Eqs. (3.19) + (3.24), Section 3.4
# --------------------------------------------------------------------------------------------
def _spectral_derivative(f):
    M = f.size
    k = np.fft.fftfreq(M, d=1.0 / M)
    if M % 2 == 0:
        k[M // 2] = 0.0
    return np.real(np.fft.ifft(1j * k * np.fft.fft(f)))


def test_p9_hilbert_transform_symbol():
    """Eq. (3.22): H cos(k.) = sin(k.), H sin(k.) = -cos(k.), H 1 = 0 (symbol -i sgn k);
    and against the principal-value integral itself by the alternating-point trapezoid rule."""
    for M in (64, 45):
        a = 2 * np.pi * np.arange(M) / M
        for k in (1, 3, 11):
            assert np.max(np.abs(oracle.hilbert(np.cos(k * a)) - np.sin(k * a))) < 1e-13
            assert np.max(np.abs(oracle.hilbert(np.sin(k * a)) + np.cos(k * a))) < 1e-13
        assert np.max(np.abs(oracle.hilbert(np.ones(M)))) < 1e-15
    M = 64
    a = 2 * np.pi * np.arange(M) / M
    f = np.exp(np.cos(a)) * np.sin(2 * a)
    m = 5
    odd = (np.arange(M) - m) % 2 == 1    # PV integral (1/pi) int 1/2 cot((a_m - b)/2) f(b) db on the staggered points
    pv = (2.0 / M) * np.sum(f[odd] / np.tan(0.5 * (a[m] - a[odd])))
    assert abs(oracle.hilbert(f)[m] - pv) < 1e-12


def test_p9_flat_surface_closed_forms():
    """zeta_0 = a: G_00 (regularised) vanishes identically, so Eq. (3.24) is -1/2 H omega'_0; flat bottom at -H:
    K_10(beta, alpha) = Im{1/2 cot((alpha - beta + iH)/2)} = -1/2 - sum_k e^{-kH} cos k(alpha - beta), hence
    K+_10 cos(p.) = -1/2 e^{-pH} cos(p.) and K+_10 1 = -1/2 (Fourier series of cot in the upper half plane)."""
    M0, M1, H, p = 64, 48, 1.3, 3
    geo = inputs.flat_flat(M0, M1, H)
    a0 = 2 * np.pi * np.arange(M0) / M0
    a1 = 2 * np.pi * np.arange(M1) / M1
    w = np.concatenate([np.sin(2 * a0), np.zeros(M1)])
    u = oracle.normal_velocity(geo.counts, geo.zeta, geo.dzeta, geo.d2zeta, w)
    assert np.max(np.abs(u - 0.5 * np.cos(2 * a0))) < 1e-14           # -1/2 H sin(2.) = +1/2 cos(2.)
    w = np.concatenate([np.zeros(M0), np.cos(p * a1) + 0.7])
    u = oracle.normal_velocity(geo.counts, geo.zeta, geo.dzeta, geo.d2zeta, w)
    assert np.max(np.abs(u - (-0.5 * np.exp(-p * H) * np.cos(p * a0) - 0.35))) < 1e-14


def test_p9_normal_velocity_of_a_known_potential_flow():
    """End-to-end pin of Section 3.4 (signs, the side of the Plemelj limit, the first-slot convention of K_j0(beta, alpha),
    the regularisation of G_00 and its diagonal, the weights 1/M_j): for f analytic in the fluid, solve (3.16) with
    b_0 = Re f, b_k = Im f (pin P3: then sum_j Phi_j = f, i.e. phi~ = Re f in the fluid), differentiate the densities
    spectrally, and compare  s_alpha d phi~/dn = Re{ f'(zeta_0) i zeta_0' }  (first line of Eq. (3.19))
    with the oracle's normal velocity.  Converges spectrally: checked at two resolutions."""
    def fprime(z):
        csc2 = lambda w: 1.0 / np.sin(w) ** 2
        return (1j * np.exp(1j * z) - 0.15 * csc2(0.5 * (z - (1.0 + 0.6j)))
                - 0.5 * (0.1 + 0.04j) * csc2(0.5 * (z - (-1.0j))) - 0.05j * csc2(0.5 * (z - (2.0 - 2.6j))))

    errs = []
    for scale in (1, 2):
        g = inputs.small_problem(96 * scale, 96 * scale, [64 * scale], seed=3).geometry
        # derivative of _f_poles, checked against a centred difference first
        z0 = 0.7 - 0.9j
        assert abs((_f_poles(z0 + 1e-6) - _f_poles(z0 - 1e-6)) / 2e-6 - fprime(z0)) < 1e-8
        b = inputs.rhs_analytic(g, _f_poles)
        A = _build(g)
        x, iters, relres, hist, status = oracle.gmres(A, b, 1e-14, 80, 600)
        assert status == 0
        dom = np.concatenate([_spectral_derivative(x[g.component(k)]) for k in range(g.counts.size)])
        u = oracle.normal_velocity(g.counts, g.zeta, g.dzeta, g.d2zeta, dom)
        s0 = g.component(0)
        exact = np.real(fprime(g.zeta[s0]) * 1j * g.dzeta[s0])
        errs.append(np.max(np.abs(u - exact)) / np.max(np.abs(exact)))
    assert errs[1] < 1e-9 and errs[1] < errs[0] * 1e-2 or errs[0] < 1e-11, errs


# --------------------------------------------------------------------------------------------
# P10  Appendix B (NEXT-4): stream function prescribed on the solids, circulations a_m = <1_m, omega> unknown
# --------------------------------------------------------------------------------------------
def _appendix_b_case():
    g = inputs.small_problem(96, 80, [48, 56], seed=5).geometry
    cents = [np.mean(g.zeta[g.component(k)]) for k in (2, 3)]    # a point inside each obstacle
    return g, cents


def test_p10_columns_are_the_boundary_values_of_phi_cyl():
    """The correction columns of Eq. (B.2) against Phi_cyl(z) = -i log(1 - e^{iz}) (Eq. 3.2)
    evaluated with numpy's complex log: rows on Gamma_0 take Re, rows on solids Im; weight 1/M_m; nothing outside the
    obstacle column blocks changes; and psi_cyl agrees with the form -log|1 - e^{iz}| used for right-hand sides."""
    g, cents = _appendix_b_case()
    B = _build(g, variant=1)
    AB = oracle.build_matrix_appendix_b(g.counts, g.kinds, g.zeta, g.dzeta, g.d2zeta, cents)
    D = AB - B
    s0, s1 = g.component(0), g.component(1)
    assert np.max(np.abs(D[:, s0])) == 0.0 and np.max(np.abs(D[:, s1])) == 0.0
    for o, k in enumerate((2, 3)):
        sk = g.component(k)
        Phi = -1j * np.log(1.0 - np.exp(1j * (g.zeta - cents[o])))
        col = np.where(np.arange(g.n) < g.counts[0], Phi.real, Phi.imag) / g.counts[k]
        assert np.max(np.abs(D[:, sk] - col[:, None])) < 1e-15
        assert np.max(np.abs(Phi.imag - inputs.psi_cyl(g.zeta - cents[o]))) < 1e-14


def test_p10_appendix_b_solution_from_the_pinned_system():
    """Consistency with the pinned system (3.16).  Solve A omega_A = b of (3.15) for GIVEN circulations a_m;
    then psi|_m = <1_m, omega_A>.  Prescribe exactly these psi|_m in Appendix B: b_0 = phi - V_1 xi,
    b_k = psi|_k - V_1 eta_k.  Because ker B = span{1_m}, the unique solution of (B.2) is
    omega_B = omega_A + sum_m (a_m - psi|_m) 1_m, and it returns the circulations: <1_m, omega_B> = a_m."""
    g, cents = _appendix_b_case()
    V1, a = 0.8, [0.6, -0.35]
    rng = np.random.default_rng(9)
    a0 = 2 * np.pi * np.arange(g.counts[0]) / g.counts[0]
    phi_t = 0.2 * np.cos(a0) + 0.1 * np.sin(3 * a0)                      # phi~ on Gamma_0
    bA = inputs.rhs_physical(g, V1, a, cents, phi_tilde=phi_t)
    A = _build(g)
    wA, it, rr, _, st = oracle.gmres(A, bA, 1e-14, 80, 600)
    assert st == 0
    psi = [np.mean(wA[g.component(k)]) for k in (2, 3)]
    # Appendix-B right-hand side: phi = phi~ + phi_mv on Gamma_0, so phi - V1 xi = phi~ + sum a_m phi_cyl(zeta_0 - z_m)
    s0 = g.component(0)
    bB = np.zeros(g.n)
    bB[s0] = phi_t + sum(am * (-1j * np.log(1.0 - np.exp(1j * (g.zeta[s0] - zm)))).real for am, zm in zip(a, cents))
    for k in range(1, g.counts.size):
        sk = g.component(k)
        pk = 0.0 if k == 1 else psi[k - 2]
        bB[sk] = pk - V1 * g.zeta[sk].imag
    AB = oracle.build_matrix_appendix_b(g.counts, g.kinds, g.zeta, g.dzeta, g.d2zeta, cents)
    assert np.linalg.cond(AB) < 1e3
    wB, it, rr, _, st = oracle.gmres(AB, bB, 1e-14, 80, 600)
    assert st == 0
    expect = wA.copy()
    for o, k in enumerate((2, 3)):
        expect[g.component(k)] += a[o] - psi[o]
        assert abs(np.mean(wB[g.component(k)]) - a[o]) < 1e-12          # the circulations come back
    assert np.max(np.abs(wB - expect)) < 1e-11


# --------------------------------------------------------------------------------------------
# P11  evaluation of Cauchy integrals near boundaries (NEXT-3): Eq. (F.4) / (5.5)
# --------------------------------------------------------------------------------------------
def _near_boundary_points(g):
    """interior points, points at distance 1e-2 ... 1e-9 from the boundaries along the inward normal, and two nodes"""
    pts = list(_interior_points())
    for k, m, sign in [(0, 7, 1.0), (1, 11, 1.0), (2, 5, 1.0), (0, 200, 1.0)]:
        s = g.component(k).start + m
        nrm = 1j * g.dzeta[s] / abs(g.dzeta[s])          # left normal of the parameterisation
        inward = -nrm if k == 0 else nrm                   # fluid is to the RIGHT of Gamma_0, to the left of solids
        for d in (1e-2, 1e-4, 1e-6, 1e-9):
            pts.append(g.zeta[s] + d * inward)
    return np.array(pts)


def test_p11_reproduces_an_analytic_function_up_to_the_boundary():
    """f analytic in the fluid (poles outside): Eq. (F.4) returns f(z) with spectral accuracy at interior points AND at
    points 1e-2 ... 1e-9 away from the boundary, where the plain trapezoid rule for (F.1) has O(1) error (PAPER.md:L569,
    L1162).  The sign sigma_0 = -1 on Gamma_0 is essential: with +1 the denominator of (F.4) vanishes (reading R18)."""
    g = inputs.make_config(1).geometry
    f = np.vstack([_f_poles(g.zeta), np.exp(2j * g.zeta), np.ones(g.n)])
    zp = _near_boundary_points(g)
    out = oracle.cauchy_eval(g.counts, g.kinds, g.zeta, g.dzeta, f, zp)
    assert np.max(np.abs(out[0] - _f_poles(zp))) < 5e-12
    assert np.max(np.abs(out[1] - np.exp(2j * zp))) < 5e-12
    assert np.max(np.abs(out[2] - 1.0)) < 1e-15                 # the weights lambda_km sum to one
    # the plain trapezoid rule of (F.1) at a point 1e-4 from Gamma_0 is useless; (F.4) is not
    z = zp[len(_interior_points()) + 1]
    plain = 0.0
    for k in range(3):
        sk = g.component(k)
        sig = -1.0 if k == 0 else 1.0
        plain += sig / g.counts[k] * np.sum(0.5 / np.tan(0.5 * (g.zeta[sk] - z)) * g.dzeta[sk] * f[0, sk]) / 1j
    assert abs(plain - _f_poles(z)) > 1e-2
    # wrong orientation of Gamma_0: denominator ~ 0
    D = sum((1.0 / g.counts[k]) * np.sum(0.5 / np.tan(0.5 * (g.zeta[g.component(k)] - zp[0])) * g.dzeta[g.component(k)])
            for k in range(3))
    assert abs(D) < 1e-12


def test_p11_coincidence_and_periodicity():
    g = inputs.make_config(1).geometry
    f = _f_poles(g.zeta)[None, :]
    s = [3, g.component(1).start + 9, g.component(2).start + 40]
    out = oracle.cauchy_eval(g.counts, g.kinds, g.zeta, g.dzeta, f, g.zeta[s])
    assert np.array_equal(out[0], f[0, s])
    zp = _interior_points()
    a = oracle.cauchy_eval(g.counts, g.kinds, g.zeta, g.dzeta, f, zp)
    b = oracle.cauchy_eval(g.counts, g.kinds, g.zeta, g.dzeta, f, zp + 2 * np.pi)
    assert np.max(np.abs(a - b)) < 1e-13                          # sum over periodic images, Eq. (3.4)
