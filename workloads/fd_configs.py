"""Seeded synthetic inputs shaped like the paper's FD-mode workloads (BASELINE.json `configs`).

This module serves BOTH the CPU oracle and the CUDA path and therefore holds none of the
method's arithmetic: no stencil coefficients, no boundary handling, no operator.  It only draws
wave functions psi[nbands,nx,ny,nz] and a local potential v_eff[nx,ny,nz] with numpy's PCG64.

The paper (PAPER.md, a review) measures this path on no public dataset, so these inputs are
synthetic stand-ins with the shapes / value distributions BASELINE.json dictates: default-like
grid spacing ~0.2 Angstrom ("lowering of the grid spacing"), molecule in a box with
zero boundaries, bulk periodic cell, k-point with Bloch phases (Eq. 13,
PAPER.md:225), slab periodic in x,y.  Recipe details not fixed by BASELINE.json are stated in
DESIGN.md ("Input recipe").

Reproducibility rule: band b of a config is drawn from default_rng([seed, b]) and v_eff from
default_rng([seed, V_STREAM]), so any subset of bands can be regenerated without the others
(needed for the 9.7 GB config 5, which is generated and checked in band chunks).
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Iterable, Optional, Sequence, Tuple

import numpy as np

BOHR_IN_ANGSTROM = 0.529177210903  # CODATA 2018; h in Bohr = h in Angstrom / this
BC_ZERO = 0
BC_PERIODIC = 1
V_STREAM = 1_000_003  # spawn key of the v_eff stream (not a band index)
BASE_SEED = 231014776


@dataclass(frozen=True)
class FDConfig:
    name: str
    index: int                      # 1-based position in BASELINE.json `configs`
    shape: Tuple[int, int, int]
    h_angstrom: Tuple[float, float, float]
    nn: int
    bc: Tuple[int, int, int]
    k: Tuple[float, float, float]   # reduced coordinates
    complex: bool
    nbands: int
    psi_kind: str                   # "normal" | "normal_envelope"
    v_kind: str                     # "uniform" | "wells_box" | "uniform_smoothed" | "wells_slab_ramp"
    v_args: Tuple[float, ...] = ()

    @property
    def seed(self) -> int:
        return BASE_SEED + self.index

    @property
    def h(self) -> Tuple[float, float, float]:
        """Grid spacings in Bohr (atomic units, as Eq. 6 is written)."""
        return tuple(x / BOHR_IN_ANGSTROM for x in self.h_angstrom)

    @property
    def dtype(self):
        return np.complex128 if self.complex else np.float64

    @property
    def npoints(self) -> int:
        return self.shape[0] * self.shape[1] * self.shape[2]

    @property
    def elem_bytes(self) -> int:
        return 16 if self.complex else 8

    @property
    def min_bytes(self) -> int:
        """Algorithmic minimum HBM traffic of one apply: read psi + write H psi + read v_eff once."""
        return 2 * self.npoints * self.nbands * self.elem_bytes + 8 * self.npoints

    def with_bands(self, nbands: int) -> "FDConfig":
        return FDConfig(**{**self.__dict__, "nbands": int(nbands)})


CONFIGS = {
    c.name: c for c in [
        FDConfig("cfg1_24c_periodic_f64", 1, (24, 24, 24), (0.2, 0.2, 0.2), 3,
                 (BC_PERIODIC,) * 3, (0.0, 0.0, 0.0), False, 8, "normal", "uniform", (-1.0, 0.0)),
        FDConfig("cfg2_48c_zero_f64", 2, (48, 48, 48), (0.18, 0.18, 0.18), 3,
                 (BC_ZERO,) * 3, (0.0, 0.0, 0.0), False, 64, "normal_envelope", "wells_box",
                 (10, 1.0, 5.0, 0.5)),
        FDConfig("cfg3_96c_periodic_f64", 3, (96, 96, 96), (0.2, 0.2, 0.2), 3,
                 (BC_PERIODIC,) * 3, (0.0, 0.0, 0.0), False, 256, "normal", "uniform_smoothed",
                 (-2.0, 0.5)),
        FDConfig("cfg4_72c_bloch_c128", 4, (72, 72, 72), (0.19, 0.19, 0.19), 3,
                 (BC_PERIODIC,) * 3, (0.25, 0.125, 0.0), True, 128, "normal", "uniform",
                 (-1.0, 0.0)),
        FDConfig("cfg5_slab_128x128x192_f64", 5, (128, 128, 192), (0.2, 0.2, 0.18), 3,
                 (BC_PERIODIC, BC_PERIODIC, BC_ZERO), (0.0, 0.0, 0.0), False, 384, "normal",
                 "wells_slab_ramp", (8, 1.0, 5.0, 0.6)),
    ]
}
CONFIG_LIST = list(CONFIGS.values())


def get(name_or_index) -> FDConfig:
    if isinstance(name_or_index, int):
        return CONFIG_LIST[name_or_index - 1]
    if name_or_index in CONFIGS:
        return CONFIGS[name_or_index]
    for c in CONFIG_LIST:
        if c.name.startswith(str(name_or_index)):
            return c
    raise KeyError(name_or_index)


def axis_coords(cfg: FDConfig, d: int) -> Tuple[np.ndarray, float]:
    """Coordinates (Bohr) of the stored points along axis d and the cell length L_d.

    Periodic: x_i = i h, L = n h.  Zero-BC: x_i = (i+1) h, L = (n+1) h (the stored array holds the
    interior points; the wave function vanishes at 0 and L).  Used by input generators only.
    """
    n, h = cfg.shape[d], cfg.h[d]
    if cfg.bc[d] == BC_PERIODIC:
        return np.arange(n) * h, n * h
    return (np.arange(n) + 1.0) * h, (n + 1) * h


def _rng(cfg: FDConfig, key: int) -> np.random.Generator:
    return np.random.default_rng([cfg.seed, int(key)])


def make_psi(cfg: FDConfig, bands: Optional[Iterable[int]] = None) -> np.ndarray:
    """psi for the listed bands (default: all), shape [len(bands), nx, ny, nz], C-contiguous."""
    bands = list(range(cfg.nbands)) if bands is None else [int(b) for b in bands]
    out = np.empty((len(bands),) + cfg.shape, dtype=cfg.dtype)
    env = None
    if cfg.psi_kind == "normal_envelope":
        # Gaussian envelope centred in the box, sigma = L/6 per axis
        g = []
        for d in range(3):
            x, L = axis_coords(cfg, d)
            g.append(np.exp(-((x - 0.5 * L) ** 2) / (2.0 * (L / 6.0) ** 2)))
        env = g[0][:, None, None] * g[1][None, :, None] * g[2][None, None, :]
    for i, b in enumerate(bands):
        r = _rng(cfg, b)
        if cfg.complex:
            re = r.standard_normal(cfg.shape)
            im = r.standard_normal(cfg.shape)
            out[i] = re + 1j * im
        else:
            out[i] = r.standard_normal(cfg.shape)
        if env is not None:
            out[i] *= env
    return out


def _wells(cfg: FDConfig, r: np.random.Generator, nwells: int, dmin: float, dmax: float,
           width_angstrom: float, lo: float, hi: float) -> np.ndarray:
    """-sum_i D_i exp(-|r-R_i|^2 / (2 w^2)); minimum image on periodic axes."""
    w = width_angstrom / BOHR_IN_ANGSTROM
    depth = r.uniform(dmin, dmax, size=nwells)
    frac = r.uniform(lo, hi, size=(nwells, 3))
    v = np.zeros(cfg.shape, dtype=np.float64)
    for i in range(nwells):
        g = []
        for d in range(3):
            x, L = axis_coords(cfg, d)
            dx = x - frac[i, d] * L
            if cfg.bc[d] == BC_PERIODIC:
                dx -= L * np.round(dx / L)
            g.append(np.exp(-(dx ** 2) / (2.0 * w * w)))
        v -= depth[i] * (g[0][:, None, None] * g[1][None, :, None] * g[2][None, None, :])
    return v


def make_veff(cfg: FDConfig) -> np.ndarray:
    """Real local potential v_eff[nx,ny,nz] in Hartree."""
    r = _rng(cfg, V_STREAM)
    if cfg.v_kind == "uniform":
        lo, hi = cfg.v_args
        return r.uniform(lo, hi, size=cfg.shape)
    if cfg.v_kind == "uniform_smoothed":
        lo, hi = cfg.v_args
        v = r.uniform(lo, hi, size=cfg.shape)
        for ax in range(3):  # 3-point box mean per axis, periodic wrap
            v = (np.roll(v, 1, axis=ax) + v + np.roll(v, -1, axis=ax)) / 3.0
        return np.ascontiguousarray(v)
    if cfg.v_kind == "wells_box":
        n, dmin, dmax, width = cfg.v_args
        return _wells(cfg, r, int(n), dmin, dmax, width, 0.2, 0.8)
    if cfg.v_kind == "wells_slab_ramp":
        n, dmin, dmax, width = cfg.v_args
        v = _wells(cfg, r, int(n), dmin, dmax, width, 0.2, 0.8)
        z, Lz = axis_coords(cfg, 2)
        return v + ((z / Lz) - 0.5)[None, None, :] * 1.0
    raise ValueError(cfg.v_kind)


def custom(shape: Sequence[int], h_angstrom: Sequence[float], bc: Sequence[int],
           k: Sequence[float] = (0.0, 0.0, 0.0), complex_: bool = False, nbands: int = 2,
           nn: int = 3, index: int = 99, name: str = "custom") -> FDConfig:
    """Ad-hoc config for shape sweeps in the tests: N(0,1) psi, U(-1,0) v_eff."""
    return FDConfig(name, index, tuple(int(s) for s in shape),
                    tuple(float(x) for x in h_angstrom), int(nn), tuple(int(b) for b in bc),
                    tuple(float(x) for x in k), bool(complex_), int(nbands), "normal", "uniform",
                    (-1.0, 0.0))
