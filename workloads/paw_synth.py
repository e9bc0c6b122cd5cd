"""Synthetic localised projector functions for the PAW non-local term.

Real PAW data sets are not available, so this module draws stand-ins
with the structure the term has in GPAW's FD mode: per atom a small box of grid points around the
atom, a handful of smooth functions p~^a_i that vanish at the box edge (s-, p-, d-like: a Gaussian
times monomials up to degree 2), and a small symmetric matrix per atom (Delta H or Delta S).  It
serves both the oracle and the CUDA path and holds none of the method's arithmetic (no
projection, no operator): only array generation.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List

import numpy as np

from .fd_configs import BC_PERIODIC, FDConfig

PAW_STREAM = 2_000_003
_MONOMIALS = [(0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), (1, 1, 0), (1, 0, 1), (0, 1, 1),
              (2, 0, 0), (0, 2, 0), (0, 0, 2), (1, 1, 1), (2, 1, 0), (0, 2, 1)]


@dataclass
class PawSet:
    box_start: np.ndarray   # int32 [natoms, 3] first grid index of the box (may be < 0 / wrap)
    box_size: np.ndarray    # int32 [natoms, 3]
    nproj: np.ndarray       # int32 [natoms]
    proj: np.ndarray        # float64, concatenated [n_i, sx, sy, sz] per atom
    dmat: np.ndarray        # float64, concatenated [n_i, n_i] per atom (symmetric)

    @property
    def natoms(self) -> int:
        return int(self.nproj.shape[0])

    @property
    def ntot(self) -> int:
        return int(self.nproj.sum())

    def proj_of(self, a: int) -> np.ndarray:
        off = 0
        for i in range(a):
            off += int(self.nproj[i]) * int(np.prod(self.box_size[i]))
        n = int(self.nproj[a]) * int(np.prod(self.box_size[a]))
        return self.proj[off:off + n].reshape((int(self.nproj[a]),) + tuple(self.box_size[a]))

    def dmat_of(self, a: int) -> np.ndarray:
        off = int(sum(int(x) ** 2 for x in self.nproj[:a]))
        n = int(self.nproj[a])
        return self.dmat[off:off + n * n].reshape(n, n)


def make_paw(cfg: FDConfig, natoms: int, nproj: int = 5, radius_angstrom: float = 0.9,
             symmetric: bool = True, vary: bool = True) -> PawSet:
    """natoms boxes at seeded positions; each axis of a box spans |x - R| <= radius.  With `vary`
    atoms alternate between nproj and max(1, nproj - 2) functions and two radii, like a compound."""
    r = np.random.default_rng([cfg.seed, PAW_STREAM])
    starts, sizes, counts, projs, dmats = [], [], [], [], []
    for a in range(natoms):
        ni = nproj if (not vary or a % 2 == 0) else max(1, nproj - 2)
        rad = (radius_angstrom if (not vary or a % 3) else 0.8 * radius_angstrom)
        centre, half = [], []
        for d in range(3):
            hd = cfg.h[d]
            rc = rad / 0.529177210903
            m = max(1, int(np.floor(rc / hd)))
            c = r.uniform(0.0, cfg.shape[d])      # fractional grid index of the atom
            centre.append(c)
            half.append(m)
        s0 = [int(np.floor(centre[d])) - half[d] + 1 for d in range(3)]
        sz = [2 * half[d] for d in range(3)]
        ax = []
        for d in range(3):
            x = (np.arange(s0[d], s0[d] + sz[d]) - centre[d]) / half[d]   # in (-1, 1)
            ax.append(x)
        X, Y, Z = np.meshgrid(*ax, indexing="ij")
        r2 = X * X + Y * Y + Z * Z
        env = np.where(r2 < 1.0, np.exp(-4.0 * r2) * (1.0 - r2) ** 2, 0.0)
        p = np.empty((ni,) + tuple(sz))
        for i in range(ni):
            ex = _MONOMIALS[i % len(_MONOMIALS)]
            p[i] = env * (X ** ex[0]) * (Y ** ex[1]) * (Z ** ex[2]) * (1.0 + 0.1 * (i // len(_MONOMIALS)))
        dm = r.uniform(-1.0, 1.0, size=(ni, ni))
        if symmetric:
            dm = 0.5 * (dm + dm.T)
        starts.append(s0)
        sizes.append(sz)
        counts.append(ni)
        projs.append(p.ravel())
        dmats.append(dm.ravel())
    return PawSet(np.array(starts, dtype=np.int32).reshape(-1, 3),
                  np.array(sizes, dtype=np.int32).reshape(-1, 3),
                  np.array(counts, dtype=np.int32),
                  np.concatenate(projs) if projs else np.zeros(0),
                  np.concatenate(dmats) if dmats else np.zeros(0))
