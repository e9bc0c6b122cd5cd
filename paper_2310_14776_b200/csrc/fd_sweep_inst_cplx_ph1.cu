// Instantiations of the sweep kernel for complex128, Bloch-phase code PH = 1 (bit 0: x/y wraps,
// bit 1: z wraps); one translation unit of several: see build.py.
#include "fd_sweep_kernel.cuh"

namespace {
template <bool HAS_V>
FdSweepKernelFn pick(int rowd)
{
    // row lengths (doubles per z row = 2 nz) with a compile-time specialisation; else run time
    switch (rowd) {
    case 48: return fd_sweep_kernel<true, HAS_V, 48, 1>;
    case 96: return fd_sweep_kernel<true, HAS_V, 96, 1>;
    case 144: return fd_sweep_kernel<true, HAS_V, 144, 1>;
    case 192: return fd_sweep_kernel<true, HAS_V, 192, 1>;
    default: return fd_sweep_kernel<true, HAS_V, 0, 1>;
    }
}
}  // namespace

FdSweepKernelFn fd_sweep_pick_cplx_ph1(int rowd, int has_v) { return has_v ? pick<true>(rowd) : pick<false>(rowd); }
