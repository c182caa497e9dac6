"""Seeded synthetic input generators (geometry + right-hand sides).

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path.  It holds
none of the method's arithmetic (no cot kernel, no matrix, no Krylov step): it only
produces the node data ``zeta, zeta', zeta''`` per boundary component, the component
tables ``counts``/``kinds`` and a right-hand side ``b``.  Arrays are generated once
and handed identically to both sides.

Shapes and sizes follow BASELINE.json ``configs`` and SURVEY.md section 8(d); they
stand in for the paper's problems 1-4 (PAPER.md:L689-L703 ellipse table (7.1),
L723 grid sizes, L795-L806 Table 3), which need the full time stepper.

Conventions (section 2): component 0 = free surface Gamma_0 (left to
right, fluid on its right), component 1 = bottom Gamma_1 (left to right, fluid on
its left), components 2.. = obstacles, parameterised CLOCKWISE (fluid on the left).
Nodes are alpha_{kl} = 2 pi l / M_k.

Right-hand side (input side of Eq. (3.15)): b_0 = phi~,
b_k = -psi_mv(zeta_k), psi_mv = V_1 eta + sum_j a_j psi_cyl(. - z_j),
psi_cyl(z) = -ln|1 - e^{iz}| (Eq. (3.2)).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Sequence

import numpy as np

KIND_SURFACE = 0
KIND_BOTTOM = 1
KIND_OBSTACLE = 2

SEED_BASE = 20210800


# --------------------------------------------------------------------------------------
# random real trigonometric series  g(a) = sum_{k=k0}^{k0+K-1} 2 Re(c_k e^{ika})
# --------------------------------------------------------------------------------------
@dataclass
class Series:
    """Real 2pi-periodic series g(a) = sum_k 2 Re(c_k e^{i k a}), k = ks[0..K-1]."""

    ks: np.ndarray  # integer wavenumbers (float64 array)
    c: np.ndarray  # complex coefficients

    def _phase(self, a: np.ndarray) -> np.ndarray:
        return np.exp(1j * np.outer(np.asarray(a, dtype=np.float64), self.ks))

    def eval(self, a, deriv: int = 0) -> np.ndarray:
        a = np.asarray(a, dtype=np.float64)
        out = np.empty(a.shape, dtype=np.float64)
        fac = self.c * (1j * self.ks) ** deriv
        flat = a.ravel()
        res = out.ravel()
        step = 4096
        for i in range(0, flat.size, step):
            res[i:i + step] = 2.0 * np.real(self._phase(flat[i:i + step]) @ fac)
        return out

    def scaled(self, s: float) -> "Series":
        return Series(self.ks.copy(), self.c * s)

    def plus(self, other: "Series") -> "Series":
        return Series(np.concatenate([self.ks, other.ks]), np.concatenate([self.c, other.c]))

    def max_abs(self, ngrid: int = 65536) -> float:
        a = 2.0 * np.pi * np.arange(ngrid) / ngrid
        return float(np.max(np.abs(self.eval(a))))


def random_series(rng: np.random.Generator, K: int, D: float, k0: int = 1,
                  amplitude: Optional[float] = None, scale: float = 1.0) -> Series:
    """c_k = scale * (a_k + i b_k) e^{-k/D}; a ~ N(0,1)^K drawn first, then b ~ N(0,1)^K.
    If ``amplitude`` is given the series is rescaled so max|g| = amplitude on a 65536 grid."""
    ks = np.arange(k0, k0 + K, dtype=np.float64)
    a = rng.standard_normal(K)
    b = rng.standard_normal(K)
    s = Series(ks, scale * (a + 1j * b) * np.exp(-ks / D))
    if amplitude is not None:
        s = s.scaled(amplitude / s.max_abs())
    return s


# --------------------------------------------------------------------------------------
# curves
# --------------------------------------------------------------------------------------
def _alpha(M: int) -> np.ndarray:
    return 2.0 * np.pi * np.arange(M) / M


def graph_curve(M: int, y0: float, g: Optional[Series]):
    """zeta = a + i (y0 + g(a)); zeta' = 1 + i g'; zeta'' = i g''."""
    a = _alpha(M)
    if g is None:
        z = a + 1j * y0
        return z, np.ones(M, dtype=np.complex128), np.zeros(M, dtype=np.complex128)
    return (a + 1j * (y0 + g.eval(a)),
            1.0 + 1j * g.eval(a, 1),
            1j * g.eval(a, 2))


def arclength_graph_curve(M: int, g: Series, ngrid: int = 1 << 18):
    """Graph y = g(x) re-parameterised so that |zeta'| = L/2pi (arclength-equispaced nodes).

    s(x) = int_0^x sqrt(1+g'^2): spectral antiderivative on ``ngrid`` points + periodic cubic
    spline; s(x_m) = L a_m / 2pi solved by Newton (stop |dx| < 1e-14)."""
    from scipy.interpolate import CubicSpline

    xg = 2.0 * np.pi * np.arange(ngrid) / ngrid
    f = np.sqrt(1.0 + g.eval(xg, 1) ** 2)
    fh = np.fft.rfft(f) / ngrid
    fbar = fh[0].real
    L = 2.0 * np.pi * fbar
    k = np.arange(fh.size, dtype=np.float64)
    ph = np.zeros_like(fh)
    ph[1:] = fh[1:] / (1j * k[1:])
    if ngrid % 2 == 0:
        ph[-1] = 0.0
    per = np.fft.irfft(ph * ngrid, n=ngrid)
    per -= per[0]  # s(0) = 0
    spl = CubicSpline(np.append(xg, 2.0 * np.pi), np.append(per, per[0]), bc_type="periodic")

    def s_of(x):
        return fbar * x + spl(np.mod(x, 2.0 * np.pi))

    a = _alpha(M)
    target = fbar * a
    # inverse-interpolation start
    sg = fbar * xg + per
    x = np.interp(target, np.append(sg, L), np.append(xg, 2.0 * np.pi))
    for _ in range(50):
        fx = np.sqrt(1.0 + g.eval(x, 1) ** 2)
        dx = (s_of(x) - target) / fx
        x = x - dx
        if np.max(np.abs(dx)) < 1e-14:
            break
    g0, g1, g2 = g.eval(x), g.eval(x, 1), g.eval(x, 2)
    w = 1.0 + g1 * g1
    x1 = fbar / np.sqrt(w)
    x2 = -fbar * g1 * g2 * x1 / w ** 1.5
    zeta = x + 1j * g0
    dzeta = (1.0 + 1j * g1) * x1
    d2zeta = 1j * g2 * x1 * x1 + (1.0 + 1j * g1) * x2
    return zeta, dzeta, d2zeta


def ellipse_curve(M: int, center: complex, q: float, b: float, tilt: float):
    """Clockwise ellipse zeta = z_j + e^{i tilt}(q cos a - i b sin a) (fluid on the left;
    PAPER.md:L89; the printed counter-clockwise form at L723 contradicts L89 -- DESIGN.md R1)."""
    a = _alpha(M)
    rot = np.exp(1j * tilt)
    return (center + rot * (q * np.cos(a) - 1j * b * np.sin(a)),
            rot * (-q * np.sin(a) - 1j * b * np.cos(a)),
            rot * (-q * np.cos(a) + 1j * b * np.sin(a)))


# --------------------------------------------------------------------------------------
# problem container
# --------------------------------------------------------------------------------------
@dataclass
class Geometry:
    counts: np.ndarray  # int32 [ncomp]
    kinds: np.ndarray  # int32 [ncomp]
    zeta: np.ndarray  # complex128 [n]
    dzeta: np.ndarray
    d2zeta: np.ndarray

    @property
    def n(self) -> int:
        return int(self.counts.sum())

    @property
    def offsets(self) -> np.ndarray:
        return np.concatenate([[0], np.cumsum(self.counts)]).astype(np.int64)

    def component(self, k: int) -> slice:
        o = self.offsets
        return slice(int(o[k]), int(o[k + 1]))


@dataclass
class Problem:
    name: str
    config: int
    stages: List[Geometry]
    rhs: List[np.ndarray]  # one right-hand side per stage
    restart: int
    tol: float = 1e-13
    max_iters: int = 1000
    centers: List[complex] = field(default_factory=list)
    notes: str = ""

    @property
    def geometry(self) -> Geometry:
        return self.stages[0]

    @property
    def n(self) -> int:
        return self.stages[0].n


def assemble(parts: Sequence[tuple], kinds: Sequence[int]) -> Geometry:
    counts = np.array([p[0].size for p in parts], dtype=np.int32)
    return Geometry(
        counts=counts,
        kinds=np.asarray(kinds, dtype=np.int32),
        zeta=np.ascontiguousarray(np.concatenate([p[0] for p in parts]).astype(np.complex128)),
        dzeta=np.ascontiguousarray(np.concatenate([p[1] for p in parts]).astype(np.complex128)),
        d2zeta=np.ascontiguousarray(np.concatenate([p[2] for p in parts]).astype(np.complex128)),
    )


# --------------------------------------------------------------------------------------
# right-hand sides (input side of Eq. (3.15))
# --------------------------------------------------------------------------------------
def psi_cyl(z: np.ndarray) -> np.ndarray:
    """psi_cyl(z) = Im Phi_cyl(z) = -ln|1 - e^{iz}|."""
    return -np.log(np.abs(1.0 - np.exp(1j * z)))


def rhs_physical(geo: Geometry, V1: float, a: Sequence[float], centers: Sequence[complex],
                 phi_tilde: Optional[np.ndarray] = None) -> np.ndarray:
    """b_0 = phi~ (zero unless given); b_k = -V1 eta_k - sum_j a_j psi_cyl(zeta_k - z_j), k >= 1."""
    b = np.zeros(geo.n, dtype=np.float64)
    s0 = geo.component(0)
    if phi_tilde is not None:
        b[s0] = phi_tilde
    for k in range(1, geo.counts.size):
        sk = geo.component(k)
        zk = geo.zeta[sk]
        v = -V1 * zk.imag
        for aj, zj in zip(a, centers):
            if aj != 0.0:
                v = v - aj * psi_cyl(zk - zj)
        b[sk] = v
    return b


def rhs_analytic(geo: Geometry, f) -> np.ndarray:
    """b_0 = Re f(zeta_0), b_k = Im f(zeta_k) for a function f analytic and 2pi-periodic in the fluid."""
    b = np.empty(geo.n, dtype=np.float64)
    for k in range(geo.counts.size):
        sk = geo.component(k)
        fz = f(geo.zeta[sk])
        b[sk] = fz.real if geo.kinds[k] == KIND_SURFACE else fz.imag
    return b


def rhs_random_smooth(geo: Geometry, rng: np.random.Generator, K: int = 64, D: float = 8.0) -> np.ndarray:
    """One random smooth series (K modes, decay e^{-k/D}, amplitude 1) per component."""
    b = np.empty(geo.n, dtype=np.float64)
    for k in range(geo.counts.size):
        sk = geo.component(k)
        ser = random_series(rng, K, D, amplitude=1.0)
        b[sk] = ser.eval(_alpha(int(geo.counts[k])))
    return b


# --------------------------------------------------------------------------------------
# the five BASELINE.json configs
# --------------------------------------------------------------------------------------
def _kinds(nobs: int):
    return [KIND_SURFACE, KIND_BOTTOM] + [KIND_OBSTACLE] * nobs


def config1() -> Problem:
    rng = np.random.default_rng(SEED_BASE + 1)
    ks = np.arange(2, 9, dtype=np.float64)
    a = rng.standard_normal(7)
    b = rng.standard_normal(7)
    eta = Series(np.array([1.0]), np.array([0.05 + 0j])).plus(
        Series(ks, 0.02 * np.exp(-ks) * (a + 1j * b)))  # 0.1 cos a = 2 Re(0.05 e^{ia})
    centers = [-1.0j]
    geo = assemble([graph_curve(256, 0.0, eta),
                    graph_curve(256, -2.0, None),
                    ellipse_curve(128, centers[0], 0.4, 0.2, 0.3)], _kinds(1))
    rhs = rhs_analytic(geo, lambda z: np.exp(1j * z))
    return Problem("cfg1_n640", 1, [geo], [rhs], restart=50, centers=centers,
                   notes="analytic f=e^{iz}")


def config2() -> Problem:
    rng = np.random.default_rng(SEED_BASE + 2)
    eta = random_series(rng, 32, 4.0, amplitude=0.15)
    tilts = rng.uniform(-np.pi / 2, np.pi / 2, size=2)
    centers = [-1.2 - 0.8j, 1.2 - 0.8j]
    geo = assemble([graph_curve(1024, 0.0, eta),
                    graph_curve(512, -2.0, None)] +
                   [ellipse_curve(256, centers[j], 0.35, 0.15, tilts[j]) for j in range(2)], _kinds(2))
    rhs = rhs_random_smooth(geo, rng, 64, 8.0)
    return Problem("cfg2_n2048", 2, [geo], [rhs], restart=50, centers=centers,
                   notes="rhs = random smooth series per component")


def config3() -> Problem:
    rng = np.random.default_rng(SEED_BASE + 3)
    eta = random_series(rng, 128, 16.0, amplitude=0.25)
    tilts = rng.uniform(-np.pi / 2, np.pi / 2, size=3)
    centers = [-2.0 - 0.9j, 0.0 - 0.9j, 2.0 - 0.9j]
    bottom = Series(np.array([1.0, 2.0]), np.array([0.25 + 0j, -0.1j]))  # 0.5 cos a + 0.2 sin 2a
    geo = assemble([graph_curve(2048, 0.0, eta),
                    graph_curve(1024, -2.0, bottom)] +
                   [ellipse_curve(512, centers[j], 0.3, 0.12, tilts[j]) for j in range(3)], _kinds(3))
    rhs = rhs_physical(geo, 1.0, [1.0, 0.0, 0.0], centers)
    return Problem("cfg3_n4608", 3, [geo], [rhs], restart=50, centers=centers,
                   notes="physical rhs (3.15), V1=1, a=(1,0,0)")


def config4(nstages: int = 4) -> Problem:
    rng = np.random.default_rng(SEED_BASE + 4)
    eta = random_series(rng, 256, 32.0, amplitude=0.4)
    bot = random_series(rng, 16, 4.0, amplitude=0.3)
    tilts = rng.uniform(-np.pi / 2, np.pi / 2, size=3)
    pert = random_series(rng, 8, 2.0, amplitude=1.0)
    centers = [-2.0 - 0.9j, 0.0 - 0.9j, 2.0 - 0.9j]
    solids = [graph_curve(2048, -2.0, bot)] + \
             [ellipse_curve(1024, centers[j], 0.3, 0.12, tilts[j]) for j in range(3)]
    stages, rhs = [], []
    for s in range(nstages):
        eta_s = eta if s == 0 else eta.plus(pert.scaled(1e-3 * s))
        geo = assemble([arclength_graph_curve(4096, eta_s)] + solids, _kinds(3))
        stages.append(geo)
        rhs.append(rhs_physical(geo, 1.0, [1.0, 0.0, 0.0], centers))
    return Problem("cfg4_n9216", 4, stages, rhs, restart=100, centers=centers,
                   notes="4 RK-like stages, Gamma_0 perturbed 1e-3 per stage")


def config5() -> Problem:
    rng = np.random.default_rng(SEED_BASE + 5)
    eta = random_series(rng, 256, 32.0, amplitude=0.5)
    bot = random_series(rng, 16, 4.0, amplitude=0.3)
    tilts = rng.uniform(-np.pi / 2, np.pi / 2, size=4)
    centers = [-2.4 - 0.9j, -0.8 - 0.9j, 0.8 - 0.9j, 2.4 - 0.9j]
    geo = assemble([arclength_graph_curve(8192, eta),
                    graph_curve(4096, -2.0, bot)] +
                   [ellipse_curve(1024, centers[j], 0.3, 0.12, tilts[j]) for j in range(4)], _kinds(4))
    rhs = rhs_physical(geo, 1.0, [1.0, 0.0, 0.0, -0.5], centers)
    return Problem("cfg5_n16384", 5, [geo], [rhs], restart=100, centers=centers,
                   notes="physical rhs, a=(1,0,0,-0.5); dense and matrix-free")


_CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


def make_config(i: int) -> Problem:
    return _CONFIGS[int(i)]()


# --------------------------------------------------------------------------------------
# small generic geometries for tests (ragged sizes, no obstacle, flat/flat, ...)
# --------------------------------------------------------------------------------------
def small_problem(M0: int, M1: int, Mobs: Sequence[int], seed: int = 7,
                  amp: float = 0.1, depth: float = 2.0) -> Problem:
    """A resolved small geometry with arbitrary (ragged) node counts."""
    rng = np.random.default_rng(seed)
    eta = random_series(rng, 4, 1.0, amplitude=amp)
    bot = random_series(rng, 3, 1.0, amplitude=0.5 * amp)
    nobs = len(Mobs)
    centers = [complex(-np.pi + 2.0 * np.pi * (j + 0.5) / max(nobs, 1), -0.5 * depth) for j in range(nobs)]
    tilts = rng.uniform(-np.pi / 2, np.pi / 2, size=nobs)
    parts = [graph_curve(M0, 0.0, eta), graph_curve(M1, -depth, bot)]
    rad = min(0.25 * depth, 0.8 * np.pi / max(nobs, 1))
    for j in range(nobs):
        parts.append(ellipse_curve(int(Mobs[j]), centers[j], rad, 0.5 * rad, tilts[j]))
    geo = assemble(parts, _kinds(nobs))
    rhs = rhs_analytic(geo, lambda z: np.exp(1j * z))
    return Problem(f"small_{M0}_{M1}_{'_'.join(map(str, Mobs))}", 0, [geo], [rhs], restart=50,
                   centers=centers)


def flat_flat(M0: int, M1: int, H: float) -> Geometry:
    """zeta_0 = a, zeta_1 = a - iH, no obstacles (textbook Fourier case)."""
    return assemble([graph_curve(M0, 0.0, None), graph_curve(M1, -H, None)], _kinds(0))
