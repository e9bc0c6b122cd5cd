"""Pins for oracle.coeffs (reading R1): textbook table, moment conditions, truncation."""
from fractions import Fraction

import numpy as np
import pytest

from helpers import golden_coeffs


@pytest.mark.parametrize("nn", [1, 2, 3, 4, 5, 6])
def test_coeffs_match_textbook_table(oracle, nn):
    want = np.array([float(c) for c in golden_coeffs()[nn]])
    got = oracle.coeffs(nn)
    assert got.shape == (nn + 1,)
    np.testing.assert_allclose(got, want, rtol=4e-16, atol=0)


def test_nn3_is_baseline_json_row(oracle):
    # BASELINE.json configs[0]: "nn=3 (coeffs -49/18, 3/2, -3/20, 1/90)"
    np.testing.assert_allclose(oracle.coeffs(3), [-49 / 18, 3 / 2, -3 / 20, 1 / 90], rtol=4e-16)


@pytest.mark.parametrize("nn", [1, 2, 3, 4, 5, 6])
def test_golden_table_satisfies_moment_conditions(nn):
    """The table itself is pinned by the order conditions of a 2nd-derivative stencil:
    sum c = 0, sum c j^2 = 2, sum c j^(2m) = 0 for m = 2..nn (exact rationals)."""
    c = golden_coeffs()[nn]
    assert c[0] + 2 * sum(c[1:]) == 0
    assert 2 * sum(c[j] * j * j for j in range(1, nn + 1)) == 2
    for m in range(2, nn + 1):
        assert sum(c[j] * Fraction(j) ** (2 * m) for j in range(1, nn + 1)) == 0


@pytest.mark.parametrize("nn", [1, 2, 3, 4, 5, 6])
def test_oracle_coeffs_moment_conditions(oracle, nn):
    c = oracle.coeffs(nn)
    j = np.arange(1, nn + 1, dtype=np.float64)
    assert abs(c[0] + 2 * c[1:].sum()) < 1e-15
    assert abs(2 * (c[1:] * j ** 2).sum() - 2) < 1e-14
    for m in range(2, nn + 1):
        assert abs((c[1:] * j ** (2 * m)).sum()) < 1e-9 * float(nn) ** (2 * m)


def test_truncation_constant_nn3(oracle):
    """First non-vanishing moment: D2 f = f'' + (h^6/560) f^(8) + ... for nn=3, so on f = x^8
    (f^(8) = 8!) the 1-D stencil error at x=0 is exactly 2 c.j^8 / 8! * 8! h^6 = h^6 * 8!/560."""
    c = golden_coeffs()[3]
    lead = 2 * sum(c[j] * Fraction(j) ** 8 for j in range(1, 4)) / Fraction(40320)
    assert lead == Fraction(1, 560)
    # and the oracle reproduces it through the operator: T = -1/2 D2 on x^8 along x, at x = 0
    n, h = 16, 0.1
    x = (np.arange(n) - 8) * h
    psi = np.broadcast_to((x ** 8)[:, None, None], (n, 7, 7)).copy()[None]
    out = oracle.apply((n, 7, 7), (h, 1.0, 1.0), 3, (0, 1, 1), None, psi)
    # y,z periodic and constant -> no contribution; x = 0 is index 8 (interior: >= 3 from faces)
    want = -0.5 * (40320.0 / 560.0) * h ** 6        # f''(0) = 0 for x^8
    assert abs(out[0, 8, 3, 3] - want) < 1e-12
    assert abs(want - (-3.6e-5)) < 1e-12            # "-3.6e-5 deviation"


def test_bad_nn_rejected(oracle):
    with pytest.raises(ValueError):
        oracle.coeffs(0)
