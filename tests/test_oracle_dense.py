"""Brute force on tiny grids: explicit dense matrix (assembled tap by tap in fd_oracle_dense, which
never calls the apply) vs the apply; vs a Kronecker-sum of 1-D band matrices built here with numpy;
spectrum vs the closed form.  SURVEY 8(c) G3, G7."""
import itertools

import numpy as np
import pytest

from helpers import coeffs_f64, planewave_eig

P, Z = 1, 0


def _t1d(n, h, bc, k, nn=3):
    """1-D kinetic matrix from the textbook table: -1/2 D2 / h^2 with wrap+phase or truncation."""
    c = coeffs_f64(nn)
    T = np.zeros((n, n), dtype=np.complex128)
    for i in range(n):
        for j in range(-nn, nn + 1):
            p = i + j
            ph = 1.0
            if p < 0 or p >= n:
                if bc == Z:
                    continue
                w = p // n
                p -= w * n
                ph = np.exp(2j * np.pi * k * w)
            T[i, p] += -0.5 * c[abs(j)] / (h * h) * ph
    return T


def _kron_sum(n, h, bc, k, v):
    Tx, Ty, Tz = [_t1d(n[d], h[d], bc[d], k[d]) for d in range(3)]
    Ix, Iy, Iz = [np.eye(n[d]) for d in range(3)]
    H = (np.kron(np.kron(Tx, Iy), Iz) + np.kron(np.kron(Ix, Ty), Iz) + np.kron(np.kron(Ix, Iy), Tz))
    if v is not None:
        H = H + np.diag(v.ravel())
    return H


@pytest.mark.parametrize("bc", list(itertools.product((Z, P), repeat=3)))
def test_dense_equals_kronecker_sum_and_apply_6cubed(oracle, bc):
    rng = np.random.default_rng(17)
    n, h = (6, 6, 6), (0.31, 0.37, 0.43)
    k = tuple(kk if b == P else 0.0 for kk, b in zip((0.25, 0.125, -0.3), bc))
    v = rng.uniform(-1, 0, n)
    M = oracle.dense(n, h, 3, bc, k, v)
    K = _kron_sum(n, h, bc, k, v)
    assert np.max(np.abs(M - K)) < 1e-12
    assert np.max(np.abs(M - M.conj().T)) < 1e-13          # Hermitian
    x = rng.standard_normal((3,) + n) + 1j * rng.standard_normal((3,) + n)
    got = oracle.apply(n, h, 3, bc, k, x, v)
    want = (M @ x.reshape(3, -1).T).T.reshape(x.shape)
    assert np.max(np.abs(got - want)) < 1e-11
    # unit vectors: column by column
    e = np.zeros((4,) + n)
    cols = [0, 43, 100, 215]
    for i, cidx in enumerate(cols):
        e[i].ravel()[cidx] = 1.0
    if all(kk == 0 for kk in k):
        cols_got = oracle.apply(n, h, 3, bc, None, e, v).reshape(4, -1)
        for i, cidx in enumerate(cols):
            assert np.max(np.abs(cols_got[i] - M[:, cidx].real)) < 1e-13


def test_dense_spectrum_is_closed_form_with_bloch(oracle):
    """on 6^3 periodic with k=(1/4,1/8,0) the 216 eigenvalues are the plane-wave values."""
    n, h, k = (6, 6, 6), (0.31, 0.37, 0.43), (0.25, 0.125, 0.0)
    M = oracle.dense(n, h, 3, (P, P, P), k, None)
    ev = np.linalg.eigvalsh(M)
    want = sorted(planewave_eig(n, h, k, m) for m in itertools.product(range(6), repeat=3))
    assert np.max(np.abs(ev - np.array(want))) < 5e-12


def test_double_hit_row_count_n_equals_2nn(oracle):
    """n_d = 2 nn periodic: taps +nn and -nn land on the same point and ADD; a 6^3 row has 16
    non-zeros, not 19."""
    M = oracle.dense((6, 6, 6), (0.3, 0.3, 0.3), 3, (P, P, P), None, None)
    nnz = (np.abs(M) > 0).sum(axis=1)
    assert set(nnz.tolist()) == {16}
    c = coeffs_f64(3)
    # the doubled entry is 2*c_3 * (-1/2 / h^2)
    assert abs(M[0, 3 * 36].real - (-0.5 * 2 * c[3] / 0.09)) < 1e-13


def test_multiple_wraps_small_axis(oracle):
    """Oracle accepts n_d < nn on a periodic axis (|w| > 1): phases exp(2 pi i k w) per wrap."""
    rng = np.random.default_rng(23)
    n, h, k = (2, 5, 1), (0.3, 0.4, 0.5), (0.2, 0.1, 0.35)
    x = rng.standard_normal((2,) + n) + 1j * rng.standard_normal((2,) + n)
    M = oracle.dense(n, h, 3, (P, P, P), k, None)
    K = _kron_sum(n, h, (P, P, P), k, None)
    assert np.max(np.abs(M - K)) < 1e-12
    got = oracle.apply(n, h, 3, (P, P, P), k, x)
    want = (M @ x.reshape(2, -1).T).T.reshape(x.shape)
    assert np.max(np.abs(got - want)) < 1e-11


def test_sines_are_not_dirichlet_eigenvectors_for_nn3(oracle):
    """SURVEY G4 trap, kept as a guard: with zero padding and nn>1 discrete sines are NOT
    eigenvectors, so nobody should 'pin' the oracle with that relation."""
    n = 12
    s = np.sin(np.pi * (np.arange(n) + 1) / (n + 1))
    psi = np.broadcast_to(s[:, None, None], (n, 4, 4)).copy()[None]
    out = oracle.apply((n, 4, 4), (1.0, 1.0, 1.0), 3, (Z, P, P), None, psi)
    ratio = out[0, :, 0, 0] / s
    assert ratio.max() - ratio.min() > 0.01
