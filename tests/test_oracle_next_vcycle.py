"""Pins of the multigrid V-cycle oracle (SURVEY 8(f) f3 completed: PAPER.md:248): the exact discrete
solution is a fixed point, cycles contract the error by a grid-independent factor, the iteration
converges to numpy's dense solve on a small zero-BC grid, the level hierarchy."""
import numpy as np
import pytest

from helpers import coeffs_f64, planewave
from test_oracle_dense import _kron_sum


def _lap_eig(n, h, m, nn):
    c = coeffs_f64(nn)
    return sum((c[0] + 2.0 * sum(c[j] * np.cos(2.0 * np.pi * m[d] / n[d] * j) for j in range(1, nn + 1)))
               / h[d] ** 2 for d in range(3))


def test_level_hierarchy(oracle):
    assert oracle.mg_levels((96, 96, 96), (1, 1, 1), 3) == [(96,) * 3, (48,) * 3, (24,) * 3, (12,) * 3,
                                                               (6,) * 3, (3,) * 3]
    assert oracle.mg_levels((31, 31, 31), (0, 0, 0), 3) == [(31,) * 3, (15,) * 3, (7,) * 3, (3,) * 3]
    assert oracle.mg_levels((32, 31, 30), (1, 0, 1), 2) == [(32, 31, 30), (16, 15, 15)]   # 15 periodic: odd
    assert oracle.mg_levels((9, 8, 8), (1, 1, 1), 3) == [(9, 8, 8)]                         # 9 periodic: odd
    assert oracle.mg_levels((16, 16, 16), (1, 1, 1), 3, max_levels=2) == [(16,) * 3, (8,) * 3]


@pytest.mark.parametrize("nn,p", [(1, 1), (3, 2), (3, 3)])
def test_exact_solution_is_a_fixed_point_and_cycles_contract(oracle, nn, p):
    n, h, bc = (16, 16, 16), (0.3, 0.25, 0.35), (1, 1, 1)
    sol = (planewave(n, (0, 0, 0), (1, 2, 0), complex_=False) +
           0.5 * planewave(n, (0, 0, 0), (3, 0, 5), complex_=False))[None]
    rhs = (_lap_eig(n, h, (1, 2, 0), nn) * planewave(n, (0, 0, 0), (1, 2, 0), complex_=False) +
           0.5 * _lap_eig(n, h, (3, 0, 5), nn) * planewave(n, (0, 0, 0), (3, 0, 5), complex_=False))[None]
    fixed = oracle.vcycle(n, h, nn, bc, p, sol, rhs)
    assert np.max(np.abs(fixed - sol)) < 1e-11
    phi = np.zeros_like(sol)
    errs = []
    for _ in range(4):
        phi = oracle.vcycle(n, h, nn, bc, p, phi, rhs)
        errs.append(np.max(np.abs(phi - sol)))
    # multigrid: a contraction per cycle well below plain Jacobi's (1 - O(h^2)): here < 0.5
    assert errs[0] < 0.5 and all(b < 0.5 * a for a, b in zip(errs, errs[1:])), errs


def test_converges_to_the_dense_solve_zero_bc(oracle):
    rng = np.random.default_rng(4)
    n, h, bc, nn, p = (7, 7, 7), (0.3, 0.33, 0.27), (0, 0, 0), 2, 2
    A = (_kron_sum_nn(n, h, bc, nn) * (1.0 / -0.5)).real        # lap_FD from the kinetic Kronecker sum
    rhs = rng.standard_normal((2,) + n)
    want = np.linalg.solve(A, rhs.reshape(2, -1).T).T.reshape(rhs.shape)
    phi = np.zeros_like(rhs)
    for _ in range(30):
        phi = oracle.vcycle(n, h, nn, bc, p, phi, rhs, nu_coarse=20)
    assert np.max(np.abs(phi - want)) < 1e-8 * np.abs(want).max()


def _kron_sum_nn(n, h, bc, nn):
    """Kronecker sum of 1-D kinetic matrices for any nn (test_oracle_dense._t1d with its nn argument)."""
    from test_oracle_dense import _t1d
    T = [_t1d(n[d], h[d], bc[d], 0.0, nn) for d in range(3)]
    I = [np.eye(n[d]) for d in range(3)]
    return (np.kron(np.kron(T[0], I[1]), I[2]) + np.kron(np.kron(I[0], T[1]), I[2]) +
            np.kron(np.kron(I[0], I[1]), T[2]))
