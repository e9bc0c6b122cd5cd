// Instantiations of the sweep kernel for float64 with real Bloch factors -1 (k_d = 1/2 on some axis:
// SURVEY 8(f) f1 "real dtype at k = 1/2"): sign flips on wrapped planes / rows / chunks, PH = 3,
// run-time row pitch only.  One translation unit of several: see build.py.
#include "fd_sweep_kernel.cuh"

namespace {
template <int MODE>
FdSweepKernelFn pick(int nn)
{
    if (nn == 1) return fd_sweep_kernel<false, MODE, 0, 3, 1, false>;
    if (nn == 2) return fd_sweep_kernel<false, MODE, 0, 3, 2, false>;
    return fd_sweep_kernel<false, MODE, 0, 3, 3, false>;
}
}  // namespace

FdSweepKernelFn fd_sweep_pick_real_ph(int mode, int nn) { return mode ? pick<1>(nn) : pick<0>(nn); }
