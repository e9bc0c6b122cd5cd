"""B200-native finite-difference Kohn-Sham apply H psi = -1/2 lap_FD psi + v_eff psi
(arXiv:2310.14776, Eq. 6 first two terms; see include/fdham.h and DESIGN.md).

The package is a thin ctypes binding over the C-ABI CUDA library libfdham.so; importing it does
not load the library (fdham.load_library() does, and raises if it has not been built).
"""
from . import fdham as _fdham
from .fdham import *  # noqa: F401,F403  (names listed in __all__ below)
from .fdham import FDError, FDHamiltonian, load_library, strerror

__all__ = [n for n in dir(_fdham) if n.startswith(("fd_", "FD"))] + ["load_library", "strerror"]
