"""Pins of fd_oracle_jacobi: the textbook 7-point update, closed-form damping of a
plane-wave mode, the fixed point, and the dense matrix form D^-1 (rhs - A phi) with zero BCs."""
import itertools

import numpy as np
import pytest

from helpers import coeffs_f64, planewave
from test_oracle_dense import _kron_sum


def _lap_eig(n, h, m, nn):
    """eigenvalue of lap_FD (scale = 1) on cos/sin plane waves of integer wave numbers m."""
    c = coeffs_f64(nn)
    lam = 0.0
    for d in range(3):
        qh = 2.0 * np.pi * m[d] / n[d]
        lam += (c[0] + 2.0 * sum(c[j] * np.cos(qh * j) for j in range(1, nn + 1))) / h[d] ** 2
    return lam


def test_seven_point_textbook_update(oracle):
    """nn = 1, omega = 1, isotropic h, periodic: phi_new = (sum of 6 neighbours - h^2 rhs) / 6."""
    rng = np.random.default_rng(2)
    n, h = (6, 7, 8), 0.3
    phi = rng.standard_normal((2,) + n)
    rhs = rng.standard_normal((2,) + n)
    got = oracle.jacobi(n, (h,) * 3, 1, (1, 1, 1), phi, rhs, 1.0, 1.0)
    nb = sum(np.roll(phi, s, axis=ax) for ax in (1, 2, 3) for s in (1, -1))
    assert np.max(np.abs(got - (nb - h * h * rhs) / 6.0)) < 1e-13


@pytest.mark.parametrize("nn", [1, 2, 3])
def test_mode_damping_and_fixed_point(oracle, nn):
    n, h = (8, 10, 12), (0.3, 0.25, 0.35)
    c = coeffs_f64(nn)
    diag = c[0] * sum(1.0 / hd ** 2 for hd in h)
    for m in [(1, 0, 0), (2, 3, 1), (4, 5, 6)]:
        mode = planewave(n, (0, 0, 0), m, complex_=False)[None]
        lam = _lap_eig(n, h, m, nn)
        for omega, scale in [(1.0, 1.0), (2.0 / 3.0, 1.0), (0.8, -0.5)]:
            out = oracle.jacobi(n, h, nn, (1, 1, 1), mode, np.zeros_like(mode), omega, scale)
            # error-propagation factor of weighted Jacobi for an eigenmode: 1 - omega lam / diag
            assert np.max(np.abs(out - (1.0 - omega * lam / diag) * mode)) < 1e-12
            # the solution of A phi = rhs is a fixed point
            out = oracle.jacobi(n, h, nn, (1, 1, 1), mode, scale * lam * mode, omega, scale)
            assert np.max(np.abs(out - mode)) < 1e-12


@pytest.mark.parametrize("bc", list(itertools.product((0, 1), repeat=3)))
def test_jacobi_matches_dense_form(oracle, bc):
    rng = np.random.default_rng(3)
    n, h, nn = (6, 6, 6), (0.31, 0.37, 0.43), 3
    phi = rng.standard_normal((2,) + n)
    rhs = rng.standard_normal((2,) + n)
    omega, scale = 0.7, 1.0
    # A = scale lap_FD = (scale / -0.5) * (kinetic Kronecker sum built from the golden table)
    A = (_kron_sum(n, h, bc, (0, 0, 0), None) * (scale / -0.5)).real
    d = np.diag(A)
    want = phi.reshape(2, -1) + omega * (rhs.reshape(2, -1) - phi.reshape(2, -1) @ A.T) / d
    got = oracle.jacobi(n, h, nn, bc, phi, rhs, omega, scale)
    assert np.max(np.abs(got.reshape(2, -1) - want)) < 1e-11
