"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

Holds no part of the method's arithmetic (see fd_configs.py).
"""
from .fd_configs import (BC_PERIODIC, BC_ZERO, BOHR_IN_ANGSTROM, CONFIG_LIST, CONFIGS, FDConfig,
                         axis_coords, custom, get, make_psi, make_veff)

from .paw_synth import PawSet, make_paw

__all__ = ["PawSet", "make_paw", "BC_PERIODIC", "BC_ZERO", "BOHR_IN_ANGSTROM", "CONFIG_LIST", "CONFIGS", "FDConfig",
           "axis_coords", "custom", "get", "make_psi", "make_veff"]
