// Instantiations of the sweep kernel for stencil half width nn = 4, complex128,
// all Bloch-phase code compiled in (PH = 3), run-time row pitch.  One translation unit of several.
#include "fd_sweep_kernel.cuh"

FdSweepKernelFn fd_sweep_pick_cplx_hi4(int mode)
{
    return mode ? fd_sweep_kernel<true, 1, 0, 3, 4, false> : fd_sweep_kernel<true, 0, 0, 3, 4, false>;
}

FdSweepKernelFn fd_sweep_pick_cplx_hi5(int mode);
FdSweepKernelFn fd_sweep_pick_cplx_hi6(int mode);
FdSweepKernelFn fd_sweep_pick_cplx_hi(int mode, int nn)
{
    if (nn == 4) return fd_sweep_pick_cplx_hi4(mode);
    if (nn == 5) return fd_sweep_pick_cplx_hi5(mode);
    return fd_sweep_pick_cplx_hi6(mode);
}
