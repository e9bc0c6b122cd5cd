"""Pins of the grid-transfer oracle: textbook weight table, moment conditions,
polynomial exactness, restriction = interpolation^T / 8, dense Kronecker brute force on all BC
mixes, constants."""
import itertools
import os
from fractions import Fraction

import numpy as np
import pytest

from helpers import GOLDEN


def golden_transfer():
    table = {}
    with open(os.path.join(GOLDEN, "transfer_weights.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            p, rest = line.split("|")
            table[int(p)] = [Fraction(t) for t in rest.split()]
    return table


def test_weights_match_textbook_table_and_moments(oracle):
    for p, row in golden_transfer().items():
        b = oracle.transfer_weights(p)
        assert b[0] == 0.0
        assert np.max(np.abs(b[1:] - np.array([float(x) for x in row]))) < 1e-15
        # exact rational moment conditions: sum 2 b_j = 1, sum b_j (j - 1/2)^(2m) = 0, m = 1..p-1
        assert 2 * sum(row) == 1
        for m in range(1, p):
            assert sum(bj * (Fraction(2 * j - 1, 2)) ** (2 * m) for j, bj in enumerate(row, 1)) == 0


def _i1d(nf, bc, p):
    """1-D interpolation matrix [nf, nc] built here from the golden table."""
    b = [0.0] + [float(x) for x in golden_transfer()[p]]
    nc = nf // 2 if bc else (nf - 1) // 2
    off = 0 if bc else 1
    M = np.zeros((nf, nc))
    for f in range(nf):
        e = f - off
        if e % 2 == 0:
            taps = [(e // 2, 1.0)]
        else:
            lo = (e - 1) // 2
            taps = [(lo - j + 1, b[j]) for j in range(1, p + 1)] + [(lo + j, b[j]) for j in range(1, p + 1)]
        for c, w in taps:
            if c < 0 or c >= nc:
                if not bc:
                    continue
                c %= nc
            M[f, c] += w
    return M


@pytest.mark.parametrize("bc", list(itertools.product((0, 1), repeat=3)))
@pytest.mark.parametrize("p", [1, 2, 3])
def test_dense_kronecker_and_adjointness(oracle, bc, p):
    rng = np.random.default_rng(11)
    nf = tuple(12 if b else 13 for b in bc)
    Ix, Iy, Iz = [_i1d(nf[d], bc[d], p) for d in range(3)]
    I3 = np.kron(np.kron(Ix, Iy), Iz)
    nc = oracle.coarse_shape(nf, bc)
    c = rng.standard_normal((2,) + nc)
    f = rng.standard_normal((2,) + nf)
    got_i = oracle.interpolate(nf, bc, p, c)
    assert np.max(np.abs(got_i.reshape(2, -1) - c.reshape(2, -1) @ I3.T)) < 1e-13
    got_r = oracle.restrict(nf, bc, p, f)
    assert np.max(np.abs(got_r.reshape(2, -1) - f.reshape(2, -1) @ I3 / 8.0)) < 1e-13
    # adjointness up to the volume ratio 8
    assert abs(8.0 * np.sum(got_r * c) - np.sum(f * got_i)) < 1e-10


@pytest.mark.parametrize("p", [1, 2, 3, 4])
def test_polynomial_exactness_in_the_interior(oracle, p):
    """degree <= 2p-1 per axis is reproduced by interpolation and sampled by restriction."""
    nf, bc = (21, 23, 25), (0, 0, 0)
    nc = oracle.coarse_shape(nf, bc)
    deg = 2 * p - 1
    xf = [np.arange(n) + 1.0 for n in nf]                     # fine coordinates, h = 1
    xc = [2.0 * (np.arange(n) + 1.0) for n in nc]             # coarse point I at fine index 2I+1
    poly = lambda X, Y, Z: (0.3 + X / 20) ** deg + (Y / 20 - 0.5) ** deg * (Z / 25) ** (deg - 1) + X * Y * Z / 4000
    F = poly(xf[0][:, None, None], xf[1][None, :, None], xf[2][None, None, :])[None]
    C = poly(xc[0][:, None, None], xc[1][None, :, None], xc[2][None, None, :])[None]
    m = 2 * p                                                  # fine points away from the walls
    gi = oracle.interpolate(nf, bc, p, C)
    assert np.max(np.abs(gi - F)[0, m:-m, m:-m, m:-m]) < 1e-12
    gr = oracle.restrict(nf, bc, p, F)
    assert np.max(np.abs(gr - C)[0, p:-p, p:-p, p:-p]) < 1e-12
    if p > 1:   # and one degree more is NOT exact (the order is what it claims to be)
        poly2 = lambda X: (X / 10.0) ** (2 * p)
        F2 = np.broadcast_to(poly2(xf[0])[:, None, None], nf)[None].copy()
        C2 = np.broadcast_to(poly2(xc[0])[:, None, None], nc)[None].copy()
        assert np.max(np.abs(oracle.interpolate(nf, bc, p, C2) - F2)[0, m:-m, m:-m, m:-m]) > 1e-9


def test_constants_and_injection_points(oracle):
    nf, bc = (8, 12, 10), (1, 1, 1)
    nc = oracle.coarse_shape(nf, bc)
    one_c = np.ones((1,) + nc)
    one_f = np.ones((1,) + nf)
    for p in (1, 2, 3):
        assert np.max(np.abs(oracle.interpolate(nf, bc, p, one_c) - 1.0)) < 1e-14
        assert np.max(np.abs(oracle.restrict(nf, bc, p, one_f) - 1.0)) < 1e-14
    rng = np.random.default_rng(0)
    c = rng.standard_normal((1,) + nc)
    f = oracle.interpolate(nf, bc, 2, c)
    assert np.max(np.abs(f[:, ::2, ::2, ::2] - c)) == 0.0      # coarse points are injected
    # zero-BC axes: coarse I sits on fine 2I+1
    nf, bc = (9, 11, 13), (0, 0, 0)
    c = rng.standard_normal((1,) + oracle.coarse_shape(nf, bc))
    f = oracle.interpolate(nf, bc, 3, c)
    assert np.max(np.abs(f[:, 1::2, 1::2, 1::2] - c)) == 0.0
    # linear interpolation next to a wall: fine 0 = (wall 0 + coarse 0) / 2
    f1 = oracle.interpolate(nf, bc, 1, c)
    assert np.max(np.abs(f1[:, 0, 1, 1] - 0.5 * c[:, 0, 0, 0])) < 1e-15
