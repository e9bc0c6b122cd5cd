"""Pins of the scaled operator `scale * lap_FD psi (+ v psi)` (a caller-supplied
prefactor instead of the -1/2 of Eq. 6; scale = 1 is the FD Laplacian of the Poisson problem).
Closed forms only -- nothing here comes from the CUDA path."""
import math

import numpy as np
import pytest

from helpers import coeffs_f64, planewave, planewave_eig

P, Z = 1, 0


@pytest.fixture(scope="module")
def oracle():
    from oracle import build, fd_oracle
    build.build()
    return fd_oracle


def test_default_scale_is_minus_one_half(oracle):
    rng = np.random.default_rng(5)
    psi = rng.standard_normal((2, 7, 8, 9))
    a = oracle.apply((7, 8, 9), (0.3, 0.25, 0.2), 3, (P, Z, P), None, psi)
    b = oracle.apply((7, 8, 9), (0.3, 0.25, 0.2), 3, (P, Z, P), None, psi, scale=-0.5)
    assert np.array_equal(a, b)


@pytest.mark.parametrize("nn", [1, 2, 3, 4])
def test_laplacian_of_a_plane_wave(oracle, nn):
    """scale = 1: lap_FD e^{iq.r} = sum_d (c_0 + 2 sum_j c_j cos(q_d j h_d)) / h_d^2 e^{iq.r}
    = -2 x the kinetic eigenvalue."""
    n, h, k, m = (8, 9, 10), (0.31, 0.27, 0.22), (0.25, 0.125, 0.0), (1, -2, 3)
    psi = planewave(n, k, m)[None]
    got = oracle.apply(n, h, nn, (P, P, P), k, psi, scale=1.0)
    lam = -2.0 * planewave_eig(n, h, k, m, nn)
    c = coeffs_f64(nn)
    direct = sum((c[0] + 2 * sum(c[j] * math.cos(2 * math.pi * (m[d] + k[d]) / n[d] * j)
                                 for j in range(1, nn + 1))) / h[d] ** 2 for d in range(3))
    assert abs(lam - direct) <= 1e-12 * abs(direct)
    assert np.max(np.abs(got - lam * psi)) <= 1e-11 * abs(lam)


def test_laplacian_of_a_quadratic_is_exact_in_the_interior(oracle):
    """lap (x^2 + 2 y^2 + 3 z^2) = 12 at points >= nn from the zero-BC faces."""
    n, h = (12, 11, 13), (0.2, 0.3, 0.25)
    x, y, z = [np.arange(n[d]) * h[d] for d in range(3)]
    f = (x[:, None, None] ** 2 + 2 * y[None, :, None] ** 2 + 3 * z[None, None, :] ** 2)[None]
    got = oracle.apply(n, h, 3, (Z, Z, Z), None, f, scale=1.0)
    assert np.max(np.abs(got[0, 3:-3, 3:-3, 3:-3] - 12.0)) <= 1e-9


def test_scale_is_linear_and_leaves_the_potential_term_alone(oracle):
    rng = np.random.default_rng(6)
    n, h = (6, 10, 8), (0.2, 0.21, 0.19)
    psi = rng.standard_normal((3,) + n) + 1j * rng.standard_normal((3,) + n)
    v = rng.uniform(-1, 0, n)
    k = (0.1, 0.0, -0.2)
    t = oracle.apply(n, h, 3, (P, Z, P), k, psi)                     # -1/2 lap
    hs = oracle.apply(n, h, 3, (P, Z, P), k, psi, v, scale=2.5)      # 2.5 lap + v
    assert np.max(np.abs(hs - (-5.0 * t + v[None] * psi))) <= 1e-10


def test_non_finite_scale_is_rejected(oracle):
    psi = np.zeros((1, 4, 4, 4))
    with pytest.raises(ValueError):
        oracle.apply((4, 4, 4), (0.2,) * 3, 3, (P, P, P), None, psi, scale=float("nan"))
