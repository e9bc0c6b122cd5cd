"""B200-native finite-difference Kohn-Sham apply H psi = -1/2 lap_FD psi + v_eff psi
(arXiv:2310.14776, Eq. 6 first two terms; see include/fdham.h and DESIGN.md).

The package is a thin ctypes binding over the C-ABI CUDA library libfdham.so; importing it does
not load the library (fdham.load_library() does, and raises if it has not been built).
"""
from .fdham import (FD_BC_PERIODIC, FD_BC_ZERO, FD_C128, FD_F64, FD_KERNEL_AUTO,
                    FD_KERNEL_GENERIC, FD_KERNEL_SWEEP, FDError, FDHamiltonian,
                    fd_apply_hamiltonian, fd_apply_hamiltonian_host, fd_apply_kinetic, fd_create,
                    fd_create_scaled, fd_destroy, fd_plan_get_kernel, fd_plan_get_weights,
                    fd_plan_kernel_for, fd_plan_launches, fd_plan_set_kernel, load_library,
                    strerror)

__all__ = [n for n in dir() if n.startswith(("fd_", "FD"))] + ["load_library", "strerror"]
