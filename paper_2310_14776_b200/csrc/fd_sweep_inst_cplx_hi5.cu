// Instantiations of the sweep kernel for stencil half width nn = 5, complex128,
// all Bloch-phase code compiled in (PH = 3), run-time row pitch.  One translation unit of several.
#include "fd_sweep_kernel.cuh"

FdSweepKernelFn fd_sweep_pick_cplx_hi5(int mode)
{
    return mode ? fd_sweep_kernel<true, 1, 0, 3, 5, false> : fd_sweep_kernel<true, 0, 0, 3, 5, false>;
}
