"""Pins of the oracle apply against what the mathematics fixes (no GPU, no stored oracle output).

Each test is aimed at one plausible mistake: wrong prefactor, wrong h axis, wrong Bloch sign,
missing wrap, non-zero padding, dropped tap, transposed axis, v_eff on the wrong operand.
"""
import os

import mpmath
import numpy as np
import pytest

from helpers import BOHR, GOLDEN, golden_coeffs, kinetic_row_sum, planewave, planewave_eig

P, Z = 1, 0


def _golden_rows():
    rows = []
    with open(os.path.join(GOLDEN, "planewave_eigs.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            n, h, k, m, lam = [t.split() for t in line.split("|")]
            rows.append((tuple(int(x) for x in n), tuple(float(x) for x in h),
                         tuple(float(x) for x in k), tuple(int(x) for x in m), lam[0]))
    return rows


@pytest.mark.parametrize("row", _golden_rows(), ids=lambda r: f"n{r[0][0]}m{r[3]}")
def test_golden_planewave_eigs_rederived_with_mpmath(row):
    """The stored values equal the closed form at 40 digits."""
    n, h_ang, k, m, lam_txt = row
    mpmath.mp.dps = 40
    c = [mpmath.mpf(x.numerator) / x.denominator for x in golden_coeffs()[3]]
    a0 = mpmath.mpf("0.529177210903")
    lam = mpmath.mpf(0)
    for d in range(3):
        hd = mpmath.mpf(repr(h_ang[d])) / a0
        qh = 2 * mpmath.pi * (m[d] + mpmath.mpf(repr(k[d]))) / n[d]
        lam += -(c[0] + 2 * sum(c[j] * mpmath.cos(qh * j) for j in (1, 2, 3))) / (2 * hd * hd)
    assert abs(lam - mpmath.mpf(lam_txt)) < mpmath.mpf(10) ** -15 * max(1, abs(lam))
    # and the double-precision closed form used elsewhere in the tests agrees with it
    h = tuple(x / BOHR for x in h_ang)
    assert abs(planewave_eig(n, h, k, m) - float(lam)) < 1e-13 * max(1.0, abs(float(lam)))


@pytest.mark.parametrize("row", [r for r in _golden_rows() if r[0][0] <= 24],
                         ids=lambda r: f"m{r[3]}")
def test_oracle_planewave_golden_small(oracle, row):
    n, h_ang, k, m, lam_txt = row
    h = tuple(x / BOHR for x in h_ang)
    psi = planewave(n, k, m)[None]
    out = oracle.apply(n, h, 3, (P, P, P), k, psi)
    lam = float(lam_txt)
    assert np.max(np.abs(out - lam * psi)) < 1e-12 * kinetic_row_sum(h)


def test_planewave_bloch_anisotropic(oracle):
    """8x9x10 anisotropic grid, k = (1/4, 1/8, 0): T psi = lambda psi."""
    n, h, k = (8, 9, 10), (0.31, 0.37, 0.43), (0.25, 0.125, 0.0)
    for m in [(0, 0, 0), (1, -2, 3), (-3, 4, 2)]:
        psi = planewave(n, k, m)[None]
        out = oracle.apply(n, h, 3, (P, P, P), k, psi)
        lam = planewave_eig(n, h, k, m)
        assert np.max(np.abs(out - lam * psi)) < 1e-12 * kinetic_row_sum(h)


def test_bloch_sign_is_discriminated(oracle):
    """With the phase sign flipped (k -> -k for the same array) the eigen-relation must FAIL
    by O(1): guards against a test that cannot see the sign (residual ~23.6)."""
    n, h, k = (8, 9, 10), (0.31, 0.37, 0.43), (0.25, 0.125, 0.0)
    m = (1, -2, 3)
    psi = planewave(n, k, m)[None]
    lam = planewave_eig(n, h, k, m)
    wrong = oracle.apply(n, h, 3, (P, P, P), tuple(-x for x in k), psi)
    assert np.max(np.abs(wrong - lam * psi)) > 1.0


def test_phase_periodicity_in_k(oracle):
    """M5: k and k + integer vector give the same operator."""
    rng = np.random.default_rng(5)
    n, h = (7, 6, 5), (0.3, 0.35, 0.4)
    psi = rng.standard_normal((2,) + n) + 1j * rng.standard_normal((2,) + n)
    a = oracle.apply(n, h, 3, (P, P, P), (0.25, 0.125, -0.4), psi)
    b = oracle.apply(n, h, 3, (P, P, P), (1.25, -1.875, 2.6), psi)
    assert np.max(np.abs(a - b)) < 1e-11


@pytest.mark.parametrize("nn", [1, 2, 3, 4, 6])
def test_planewave_gamma_all_orders(oracle, nn):
    n, h = (13, 12, 14), (0.3, 0.25, 0.35)
    m = (2, -1, 3)
    psi = planewave(n, (0, 0, 0), m)[None]
    out = oracle.apply(n, h, nn, (P, P, P), (0, 0, 0), psi)
    lam = planewave_eig(n, h, (0, 0, 0), m, nn)
    assert np.max(np.abs(out - lam * psi)) < 1e-12 * kinetic_row_sum(h, nn)
    # real dtype sees the same eigenvalue on cos(q.r)
    psr = np.ascontiguousarray(psi.real)
    outr = oracle.apply(n, h, nn, (P, P, P), None, psr)
    assert np.max(np.abs(outr - lam * psr)) < 1e-12 * kinetic_row_sum(h, nn)


def test_eigenvalue_converges_to_half_q2(oracle):
    """Prefactor pin: lambda -> q^2/2 (atomic units, Eq. 6 has -1/2 nabla^2) with O(h^6) error."""
    n = (24, 24, 24)
    h = (0.2 / BOHR,) * 3
    psi = planewave(n, (0, 0, 0), (1, 0, 0))[None]
    out = oracle.apply(n, h, 3, (P, P, P), None, np.ascontiguousarray(psi.real))
    lam = out[0, 0, 0, 0] / psi.real[0, 0, 0, 0]
    q = 2 * np.pi / (n[0] * h[0])
    assert abs(lam - 0.5 * q * q) < 2e-7            # 0.23991051619... vs 0.23991065266...
    assert abs(lam - 0.23991051619666738) < 1e-13


def test_constants_map_to_zero_periodic(oracle):
    n, h = (9, 10, 11), (0.2 / BOHR,) * 3
    psi = np.full((1,) + n, 3.7)
    out = oracle.apply(n, h, 3, (P, P, P), None, psi)
    assert np.max(np.abs(out)) <= 1e-13 * kinetic_row_sum(h) * 3.7


def test_constants_do_not_vanish_at_zero_bc_faces(oracle):
    """Zero padding really is zero: a constant is NOT annihilated within nn of a zero-BC face,
    and the value there is the closed-form truncated row sum."""
    n, h = (12, 5, 5), (0.5, 0.5, 0.5)
    psi = np.ones((1,) + n)
    out = oracle.apply(n, h, 3, (Z, P, P), None, psi)
    c = [float(x) for x in golden_coeffs()[3]]
    # at ix = 0: taps -1,-2,-3 are dropped -> row sum = c0 + c1 + c2 + c3
    want0 = -0.5 / 0.25 * (c[0] + c[1] + c[2] + c[3])
    want1 = -0.5 / 0.25 * (c[0] + 2 * c[1] + c[2] + c[3])
    want2 = -0.5 / 0.25 * (c[0] + 2 * c[1] + 2 * c[2] + c[3])
    np.testing.assert_allclose(out[0, 0], want0, rtol=1e-13)
    np.testing.assert_allclose(out[0, 1], want1, rtol=1e-13)
    np.testing.assert_allclose(out[0, 2], want2, rtol=1e-13)
    np.testing.assert_allclose(out[0, -1], want0, rtol=1e-13)
    assert np.max(np.abs(out[0, 3:-3])) < 1e-13


def test_polynomial_exactness_interior(oracle):
    """exact on x^a y^b z^c with a,b,c <= 2nn+1 at points >= nn from zero-BC faces."""
    n, hh = (10, 10, 10), 0.1
    x = (np.arange(10) - 4.5) * hh
    X, Y, Zc = np.meshgrid(x, x, x, indexing="ij")
    f = X ** 7 + Y ** 6 + Zc ** 7 * X ** 2
    lap = 42 * X ** 5 + 30 * Y ** 4 + 42 * Zc ** 5 * X ** 2 + 2 * Zc ** 7
    out = oracle.apply(n, (hh,) * 3, 3, (Z, Z, Z), None, f[None])
    inner = (slice(3, 7),) * 3
    assert np.max(np.abs(out[0][inner] + 0.5 * lap[inner])) < 5e-12
    # the same polynomial is NOT reproduced at the faces (zero padding), so the slice matters
    assert np.max(np.abs(out[0] + 0.5 * lap)) > 1.0


def test_polynomial_anisotropic_axes_not_swapped(oracle):
    """f = x^2 only: T f = -1 everywhere in the interior regardless of h_y, h_z; f = z^2 likewise.
    A swapped h axis or transposed array index breaks this when h differ by axis."""
    n, h = (9, 8, 11), (0.2, 0.3, 0.5)
    for ax in range(3):
        x = (np.arange(n[ax]) - 4.0) * h[ax]
        shp = [1, 1, 1]
        shp[ax] = n[ax]
        f = np.broadcast_to((x ** 2).reshape(shp), n).copy()
        bc = [P, P, P]
        bc[ax] = Z
        out = oracle.apply(n, h, 3, bc, None, f[None])
        sl = [slice(None)] * 3
        sl[ax] = slice(3, n[ax] - 3)
        assert np.max(np.abs(out[0][tuple(sl)] + 1.0)) < 1e-11


def test_hermiticity(oracle):
    rng = np.random.default_rng(11)
    # (bc, k, complex)
    cases = [((P, P, Z), None, False), ((Z, Z, Z), None, False),
             ((P, P, P), (0.25, 0.125, 0.0), True), ((P, Z, P), (0.3, 0.0, -0.2), True)]
    n, h = (7, 8, 9), (0.31, 0.37, 0.29)
    for bc, k, cplx in cases:
        v = rng.uniform(-1, 0, n)
        a = rng.standard_normal((1,) + n)
        b = rng.standard_normal((1,) + n)
        if cplx:
            a = a + 1j * rng.standard_normal((1,) + n)
            b = b + 1j * rng.standard_normal((1,) + n)
        Ha = oracle.apply(n, h, 3, bc, k, a, v)
        Hb = oracle.apply(n, h, 3, bc, k, b, v)
        lhs = np.vdot(a, Hb)
        rhs = np.vdot(Ha, b)
        assert abs(lhs - rhs) < 1e-10, (bc, k)


def test_veff_constant_shifts_eigenvalue_and_is_linear(oracle):
    n, h = (8, 8, 8), (0.3,) * 3
    m = (1, 2, -1)
    psi = planewave(n, (0, 0, 0), m)[None]
    lam = planewave_eig(n, h, (0, 0, 0), m)
    v = np.full(n, -0.75)
    out = oracle.apply(n, h, 3, (P, P, P), (0, 0, 0), psi, v)
    assert np.max(np.abs(out - (lam - 0.75) * psi)) < 1e-12 * kinetic_row_sum(h)
    rng = np.random.default_rng(3)
    v1, v2 = rng.uniform(-1, 0, n), rng.uniform(-2, 2, n)
    x = rng.standard_normal((3,) + n)
    d = oracle.apply(n, h, 3, (P, Z, P), None, x, v1 + v2) - oracle.apply(n, h, 3, (P, Z, P), None, x, v1)
    assert np.max(np.abs(d - v2[None] * x)) < 1e-12
    t0 = oracle.apply(n, h, 3, (P, Z, P), None, x, np.zeros(n))
    t1 = oracle.apply(n, h, 3, (P, Z, P), None, x)
    assert np.array_equal(t0, t1)


def test_translation_invariance_periodic(oracle):
    rng = np.random.default_rng(2)
    n, h = (7, 9, 8), (0.3, 0.2, 0.25)
    x = rng.standard_normal((2,) + n)
    base = oracle.apply(n, h, 3, (P, P, P), None, x)
    for shift, ax in [(1, 1), (3, 2), (5, 3), (-2, 1)]:
        got = oracle.apply(n, h, 3, (P, P, P), None, np.ascontiguousarray(np.roll(x, shift, axis=ax)))
        assert np.max(np.abs(got - np.roll(base, shift, axis=ax))) < 1e-11


def test_complex_gamma_equals_two_real_applies(oracle):
    rng = np.random.default_rng(8)
    n, h = (6, 7, 8), (0.3, 0.2, 0.25)
    re, im = rng.standard_normal((2, 2) + n)
    v = rng.uniform(-1, 0, n)
    c = oracle.apply(n, h, 3, (P, Z, P), (0, 0, 0), re + 1j * im, v)
    r = oracle.apply(n, h, 3, (P, Z, P), None, re, v)
    i = oracle.apply(n, h, 3, (P, Z, P), None, im, v)
    assert np.max(np.abs(c - (r + 1j * i))) < 1e-12


def test_band_independence_and_points(oracle):
    rng = np.random.default_rng(9)
    n, h = (6, 5, 7), (0.3, 0.2, 0.25)
    x = rng.standard_normal((5,) + n)
    v = rng.uniform(-1, 0, n)
    full = oracle.apply(n, h, 3, (P, P, Z), None, x, v, nthreads=3)
    for b in range(5):
        one = oracle.apply(n, h, 3, (P, P, Z), None, x[b:b + 1], v, nthreads=1)
        assert np.array_equal(one[0], full[b])
    pts = np.array([[0, 0, 0, 0], [4, 5, 4, 6], [2, 3, 0, 1]])
    got = oracle.points(n, h, 3, (P, P, Z), None, x, v, pts)
    assert np.array_equal(got, np.array([full[tuple(p)] for p in pts]))
