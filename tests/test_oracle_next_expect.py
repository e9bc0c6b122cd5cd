"""Pins of the SURVEY 8(f) f2 oracle functions (fd_oracle_expect, fd_oracle_residual): plane waves
(eps = lambda P, norm = P), Hermiticity (Im eps = 0), constant-v shift, the 6^3 dense matrix built
here from the textbook table (x^H M x), residual of an eigenvector = 0."""
import itertools

import numpy as np
import pytest

from helpers import planewave, planewave_eig
from test_oracle_dense import _kron_sum

BOHR = 0.529177210903


def test_planewave_expectation_values(oracle):
    n, h = (8, 9, 10), (0.2 / BOHR, 0.21 / BOHR, 0.18 / BOHR)
    k = (0.25, 0.125, -0.3)
    ms = [(0, 0, 0), (1, -2, 3), (3, 2, -1)]
    psi = np.stack([planewave(n, k, m) for m in ms]) * np.array([1.0, 2.0, 0.5j])[:, None, None, None]
    P = np.prod(n)
    eps, norm = oracle.expect(n, h, 3, (1, 1, 1), k, psi, None)
    amp2 = np.array([1.0, 4.0, 0.25])
    lam = np.array([planewave_eig(n, h, k, m) for m in ms])
    assert np.allclose(norm, amp2 * P, rtol=1e-13)
    assert np.max(np.abs(eps - lam * amp2 * P)) < 1e-10 * P
    # a constant potential shifts eps by v * norm
    v = np.full(n, -0.7)
    eps_v, norm_v = oracle.expect(n, h, 3, (1, 1, 1), k, psi, v)
    assert np.allclose(norm_v, norm)
    assert np.max(np.abs(eps_v - (eps - 0.7 * norm))) < 1e-10 * P


@pytest.mark.parametrize("bc", [(1, 1, 1), (0, 1, 0), (0, 0, 0), (1, 0, 1)])
def test_expect_is_real_and_matches_dense_quadratic_form(oracle, bc):
    rng = np.random.default_rng(5)
    n, h = (6, 6, 6), (0.31, 0.37, 0.43)
    k = tuple(kk if b else 0.0 for kk, b in zip((0.25, 0.125, -0.3), bc))
    v = rng.uniform(-1, 0, n)
    x = rng.standard_normal((4,) + n) + 1j * rng.standard_normal((4,) + n)
    eps, norm, out = oracle.expect(n, h, 3, bc, k, x, v, want_out=True)
    M = _kron_sum(n, h, bc, k, v)           # built in the test from the golden coefficient table
    xf = x.reshape(4, -1)
    want = np.einsum("bi,ij,bj->b", xf.conj(), M, xf)
    assert np.max(np.abs(eps - want)) < 1e-10
    assert np.max(np.abs(eps.imag)) < 1e-10                     # Hermitian operator
    assert np.allclose(norm, np.sum(np.abs(xf) ** 2, axis=1), rtol=1e-13)
    assert np.max(np.abs(out - oracle.apply(n, h, 3, bc, k, x, v))) == 0.0


def test_expect_real_dtype_and_scale(oracle):
    rng = np.random.default_rng(6)
    n, h, bc = (7, 8, 9), (0.3, 0.35, 0.4), (1, 0, 1)
    x = rng.standard_normal((3,) + n)
    v = rng.uniform(-1, 1, n)
    for scale in (-0.5, 1.0):
        eps, norm = oracle.expect(n, h, 2, bc, None, x, v, scale=scale)
        hx = oracle.apply(n, h, 2, bc, None, x, v, scale=scale)
        assert np.allclose(eps.real, np.sum(x * hx, axis=(1, 2, 3)), rtol=1e-12)
        assert np.all(eps.imag == 0.0)
        assert np.allclose(norm, np.sum(x * x, axis=(1, 2, 3)), rtol=1e-13)
    # linear in scale for the kinetic part: eps(scale) - sum v x^2 proportional to scale
    e1, _ = oracle.expect(n, h, 2, bc, None, x, None, scale=1.0)
    e2, _ = oracle.expect(n, h, 2, bc, None, x, None, scale=-0.5)
    assert np.allclose(e2.real, -0.5 * e1.real, rtol=1e-12)


def test_residual_of_eigenvector_vanishes(oracle):
    n, h, k = (8, 8, 8), (0.4, 0.4, 0.4), (0.25, 0.0, 0.125)
    ms = [(1, 0, 2), (0, 0, 0)]
    psi = np.stack([planewave(n, k, m) for m in ms])
    hpsi = oracle.apply(n, h, 3, (1, 1, 1), k, psi, None)
    eps, norm = oracle.expect(n, h, 3, (1, 1, 1), k, psi, None)
    lam = eps.real / norm
    assert np.allclose(lam, [planewave_eig(n, h, k, m) for m in ms], rtol=1e-12)
    r = oracle.residual(psi, hpsi, lam)
    assert np.max(np.abs(r)) < 1e-12 * 60
    # and of a non-eigenvector it is hpsi - lam psi, orthogonal to psi
    rng = np.random.default_rng(1)
    x = rng.standard_normal((2,) + n)
    hx = oracle.apply(n, h, 3, (1, 1, 1), None, x, None)
    e, nr = oracle.expect(n, h, 3, (1, 1, 1), None, x, None)
    rr = oracle.residual(x, hx, e.real / nr)
    assert np.max(np.abs(np.sum(rr * x, axis=(1, 2, 3)))) < 1e-9
    assert np.max(np.abs(rr - (hx - (e.real / nr)[:, None, None, None] * x))) < 1e-13
