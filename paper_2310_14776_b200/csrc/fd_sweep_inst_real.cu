// Instantiations of the sweep kernel for float64 (one translation unit of several: see build.py).
#include "fd_sweep_kernel.cuh"

namespace {
template <bool HAS_V>
FdSweepKernelFn pick(int rowd)
{
    // row lengths (doubles per z row) with a compile-time specialisation; else run-time pitch
    switch (rowd) {
    case 24: return fd_sweep_kernel<false, HAS_V, 24, 0>;
    case 48: return fd_sweep_kernel<false, HAS_V, 48, 0>;
    case 64: return fd_sweep_kernel<false, HAS_V, 64, 0>;
    case 96: return fd_sweep_kernel<false, HAS_V, 96, 0>;
    case 128: return fd_sweep_kernel<false, HAS_V, 128, 0>;
    case 192: return fd_sweep_kernel<false, HAS_V, 192, 0>;
    default: return fd_sweep_kernel<false, HAS_V, 0, 0>;
    }
}
}  // namespace

FdSweepKernelFn fd_sweep_pick_real(int rowd, int has_v) { return has_v ? pick<true>(rowd) : pick<false>(rowd); }
