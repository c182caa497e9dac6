"""The seeded input generators: shapes of BASELINE.json's configs, determinism, orientation and the
consistency zeta' = d zeta/d alpha, zeta'' = d^2 zeta/d alpha^2 (checked by FFT differentiation)."""
import numpy as np
import pytest

from paper_2108_01786_b200 import inputs

EXPECT = {1: (640, [256, 256, 128]), 2: (2048, [1024, 512, 256, 256]),
          3: (4608, [2048, 1024, 512, 512, 512])}


def _fft_derivative(f):
    M = f.size
    k = np.fft.fftfreq(M, 1.0 / M)
    if M % 2 == 0:
        k[M // 2] = 0.0
    return np.fft.ifft(1j * k * np.fft.fft(f))


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_config_shapes_and_determinism(cfg):
    P = inputs.make_config(cfg)
    Q = inputs.make_config(cfg)
    g = P.geometry
    n, counts = EXPECT[cfg]
    assert g.n == n and list(g.counts) == counts
    assert list(g.kinds) == [0, 1] + [2] * (len(counts) - 2)
    for a, b in ((g.zeta, Q.geometry.zeta), (g.dzeta, Q.geometry.dzeta), (P.rhs[0], Q.rhs[0])):
        assert np.array_equal(a, b)
    assert P.rhs[0].shape == (n,) and np.all(np.isfinite(P.rhs[0]))


@pytest.mark.parametrize("cfg", [1, 2])
def test_derivatives_are_consistent(cfg):
    g = inputs.make_config(cfg).geometry
    for k in range(g.counts.size):
        s = g.component(k)
        M = int(g.counts[k])
        a = 2 * np.pi * np.arange(M) / M
        z = g.zeta[s] - (a if g.kinds[k] != inputs.KIND_OBSTACLE else 0.0)  # periodic part
        d1 = _fft_derivative(z) + (1.0 if g.kinds[k] != inputs.KIND_OBSTACLE else 0.0)
        d2 = _fft_derivative(_fft_derivative(z))
        assert np.max(np.abs(d1 - g.dzeta[s])) < 1e-9
        assert np.max(np.abs(d2 - g.d2zeta[s])) < 1e-6


def test_orientation_and_separation():
    """Obstacles clockwise (negative signed area), graphs left to right; boundaries do not touch."""
    for cfg in (1, 2, 3):
        g = inputs.make_config(cfg).geometry
        for k in range(g.counts.size):
            s = g.component(k)
            z, dz = g.zeta[s], g.dzeta[s]
            if g.kinds[k] == inputs.KIND_OBSTACLE:
                area = 0.5 * np.sum(np.imag(np.conj(z - z.mean()) * dz)) * 2 * np.pi / z.size
                assert area < 0
            else:
                assert np.all(dz.real > 0)
        # minimal distance between different components
        for k in range(g.counts.size):
            for j in range(k + 1, g.counts.size):
                zk, zj = g.zeta[g.component(k)], g.zeta[g.component(j)]
                d = np.abs(zk[:, None] - zj[None, :])
                for sh in (-2 * np.pi, 2 * np.pi):
                    d = np.minimum(d, np.abs(zk[:, None] - zj[None, :] + sh))
                assert d.min() > 0.15


def test_arclength_curve_is_equispaced_in_arclength():
    rng = np.random.default_rng(3)
    gser = inputs.random_series(rng, 6, 2.0, amplitude=0.4)
    z, dz, d2z = inputs.arclength_graph_curve(1024, gser)
    assert np.max(np.abs(np.abs(dz) - np.abs(dz[0]))) < 1e-12
    assert np.max(np.abs(z.imag - gser.eval(z.real))) < 1e-14
    # zeta'' is the derivative of zeta' (periodic)
    assert np.max(np.abs(_fft_derivative(dz) - d2z)) < 1e-8


def test_small_problem_ragged():
    P = inputs.small_problem(37, 29, [19, 23], seed=1)
    assert P.n == 37 + 29 + 19 + 23 and P.rhs[0].shape == (P.n,)
