// Instantiations of the sweep kernel for the higher stencil orders nn = 4, 5, 6,
// float64: 2-row micro tile, general z-tap form, run-time row pitch.  One translation unit of
// several: see build.py.
#include "fd_sweep_kernel.cuh"

namespace {
template <int MODE>
FdSweepKernelFn pick(int nn)
{
    if (nn == 4) return fd_sweep_kernel<false, MODE, 0, 0, 4, false>;
    if (nn == 5) return fd_sweep_kernel<false, MODE, 0, 0, 5, false>;
    return fd_sweep_kernel<false, MODE, 0, 0, 6, false>;
}
}  // namespace

FdSweepKernelFn fd_sweep_pick_real_hi(int mode, int nn) { return mode ? pick<1>(nn) : pick<0>(nn); }
