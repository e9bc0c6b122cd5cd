// Instantiations of the sweep kernel for complex128, Bloch-phase code PH = 0 (bit 0: x/y wraps,
// bit 1: z wraps); one translation unit of several: see build.py.
#include "fd_sweep_kernel.cuh"

namespace {
template <bool HAS_V>
FdSweepKernelFn pick(int rowd, int nn)
{
    // other stencil orders: run-time row pitch only
    if (nn == 1) return fd_sweep_kernel<true, HAS_V, 0, 0, 1>;
    if (nn == 2) return fd_sweep_kernel<true, HAS_V, 0, 0, 2>;
    // nn = 3: row lengths (doubles per z row = 2 nz) with a compile-time specialisation
    switch (rowd) {
    case 48: return fd_sweep_kernel<true, HAS_V, 48, 0, 3>;
    case 96: return fd_sweep_kernel<true, HAS_V, 96, 0, 3>;
    case 144: return fd_sweep_kernel<true, HAS_V, 144, 0, 3>;
    case 192: return fd_sweep_kernel<true, HAS_V, 192, 0, 3>;
    default: return fd_sweep_kernel<true, HAS_V, 0, 0, 3>;
    }
}
}  // namespace

FdSweepKernelFn fd_sweep_pick_cplx_ph0(int rowd, int has_v, int nn)
{
    return has_v ? pick<true>(rowd, nn) : pick<false>(rowd, nn);
}
