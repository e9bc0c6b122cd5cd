// Instantiations of the sweep kernel for the weighted-Jacobi sweep (MODE 2: float64, a per-band
// right-hand side rides the second staged array); one translation unit of several: see build.py.
#include "fd_sweep_kernel.cuh"

FdSweepKernelFn fd_sweep_pick_real_jacobi(int rowd, int nn)
{
    if (nn == 1) return fd_sweep_kernel<false, 2, 0, 0, 1, false>;
    if (nn == 2) return fd_sweep_kernel<false, 2, 0, 0, 2, false>;
    switch (rowd) {
    case 48: return fd_sweep_kernel<false, 2, 48, 0, 3, false>;
    case 96: return fd_sweep_kernel<false, 2, 96, 0, 3, false>;
    case 192: return fd_sweep_kernel<false, 2, 192, 0, 3, false>;
    default: return fd_sweep_kernel<false, 2, 0, 0, 3, false>;
    }
}
