// Instantiations of the sweep kernel for float64 (one translation unit of several: see build.py).
#include "fd_sweep_kernel.cuh"

namespace {
template <bool HAS_V>
FdSweepKernelFn pick(int rowd, int nn)
{
    // other stencil orders: run-time row pitch only
    if (nn == 1) return fd_sweep_kernel<false, HAS_V, 0, 0, 1>;
    if (nn == 2) return fd_sweep_kernel<false, HAS_V, 0, 0, 2>;
    // nn = 3: row lengths (doubles per z row) with a compile-time specialisation, else run time
    switch (rowd) {
    case 24: return fd_sweep_kernel<false, HAS_V, 24, 0, 3>;
    case 48: return fd_sweep_kernel<false, HAS_V, 48, 0, 3>;
    case 64: return fd_sweep_kernel<false, HAS_V, 64, 0, 3>;
    case 96: return fd_sweep_kernel<false, HAS_V, 96, 0, 3>;
    case 128: return fd_sweep_kernel<false, HAS_V, 128, 0, 3>;
    case 192: return fd_sweep_kernel<false, HAS_V, 192, 0, 3>;
    default: return fd_sweep_kernel<false, HAS_V, 0, 0, 3>;
    }
}
}  // namespace

FdSweepKernelFn fd_sweep_pick_real(int rowd, int has_v, int nn)
{
    return has_v ? pick<true>(rowd, nn) : pick<false>(rowd, nn);
}
