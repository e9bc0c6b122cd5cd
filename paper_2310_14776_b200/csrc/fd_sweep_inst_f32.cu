// Instantiations of the sweep kernel for float32 and complex64: run-time row pitch,
// nn = 1..3, complex64 with all Bloch-phase code (PH = 3).  One translation unit of several.
#include "fd_sweep_kernel.cuh"

namespace {
template <bool CPLX, int MODE>
FdSweepKernelFn pick(int nn)
{
    constexpr int PH = CPLX ? 3 : 0;
    if (nn == 1) return fd_sweep_kernel<CPLX, MODE, 0, PH, 1, false, true>;
    if (nn == 2) return fd_sweep_kernel<CPLX, MODE, 0, PH, 2, false, true>;
    return fd_sweep_kernel<CPLX, MODE, 0, PH, 3, false, true>;
}
}  // namespace

FdSweepKernelFn fd_sweep_pick_f32(int cplx, int mode, int nn)
{
    if (cplx) return mode ? pick<true, 1>(nn) : pick<true, 0>(nn);
    return mode ? pick<false, 1>(nn) : pick<false, 0>(nn);
}
