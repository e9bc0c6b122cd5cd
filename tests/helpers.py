"""Test-side helpers: textbook coefficient table (tests/golden/fd_coeffs.txt), closed forms and
the parity tolerance.  Nothing here imports the oracle or the CUDA path."""
from __future__ import annotations

import math
import os
from fractions import Fraction

import numpy as np

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
BOHR = 0.529177210903


def golden_coeffs() -> dict:
    """{nn: [Fraction c_0..c_nn]} from tests/golden/fd_coeffs.txt (Fornberg 1988 / BASELINE.json)."""
    table = {}
    with open(os.path.join(GOLDEN, "fd_coeffs.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            nn, rest = line.split("|")
            table[int(nn)] = [Fraction(t) for t in rest.split()]
    return table


def coeffs_f64(nn: int) -> np.ndarray:
    return np.array([float(c) for c in golden_coeffs()[nn]], dtype=np.float64)


def kinetic_row_sum(h, nn: int = 3, scale: float = -0.5) -> float:
    """S = |scale| sum_d (|c_0| + 2 sum_j |c_j|) / h_d^2 : absolute row sum of scale * lap_FD; for
    the kinetic operator (scale = -1/2) this is DESIGN.md reading R10."""
    c = golden_coeffs()[nn]
    a = float(abs(c[0]) + 2 * sum(abs(x) for x in c[1:]))
    return abs(scale) * sum(a / (hd * hd) for hd in h)


def parity_tol(h, nn, psi: np.ndarray, v_eff, scale: float = -0.5) -> float:
    """north_star: max|d| <= 1e-12 (max|psi| * S + max|v_eff psi|)."""
    s = kinetic_row_sum(h, nn, scale)
    mp = float(np.max(np.abs(psi))) if psi.size else 0.0
    mv = 0.0
    if v_eff is not None and psi.size:
        mv = float(np.max(np.abs(v_eff[None] * psi)))
    return 1e-12 * (mp * s + mv)


def planewave_eig(n, h, k, m, nn: int = 3) -> float:
    """lambda = -1/2 sum_d (c_0 + 2 sum_j c_j cos(q_d j h_d)) / h_d^2 in double precision."""
    c = coeffs_f64(nn)
    lam = 0.0
    for d in range(3):
        qh = 2.0 * math.pi * (m[d] + k[d]) / n[d]
        s = c[0] + 2.0 * sum(c[j] * math.cos(qh * j) for j in range(1, nn + 1))
        lam += -0.5 * s / (h[d] * h[d])
    return lam


def planewave(n, k, m, complex_=True) -> np.ndarray:
    """exp(i sum_d 2 pi (m_d + k_d) i_d / n_d) on the grid (periodic coordinates x_i = i h)."""
    ph = [2.0 * np.pi * (m[d] + k[d]) * np.arange(n[d]) / n[d] for d in range(3)]
    arg = ph[0][:, None, None] + ph[1][None, :, None] + ph[2][None, None, :]
    return np.exp(1j * arg) if complex_ else np.cos(arg)
