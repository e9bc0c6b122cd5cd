// Generator of one instantiation unit of the sweep kernel (fd_sweep_kernel.cuh).  The including
// .cu file defines
//   FD_INST_CPLX   false | true
//   FD_INST_PH     Bloch-phase code compiled in (complex: 0, 1, 3; real: 0)
//   FD_INST_EX     false | true  (expectation-value epilogue)
//   FD_INST_NAME   name of the exported pick function
//   FD_INST_ROWS(X) X(row length in doubles) ... : nn = 3 row lengths with a compile-time pitch
// and gets  FdSweepKernelFn FD_INST_NAME(int rowd, int mode, int nn)  for mode 0 (kinetic) and 1
// (+ v_eff psi).  The units exist so that build.py can compile them in parallel.
#include "fd_sweep_kernel.cuh"

namespace {
template <int MODE>
FdSweepKernelFn pick(int rowd, int nn)
{
    // other stencil orders: run-time row pitch only
    if (nn == 1) return fd_sweep_kernel<FD_INST_CPLX, MODE, 0, FD_INST_PH, 1, FD_INST_EX>;
    if (nn == 2) return fd_sweep_kernel<FD_INST_CPLX, MODE, 0, FD_INST_PH, 2, FD_INST_EX>;
    switch (rowd) {
#define FD_INST_CASE(R) \
    case R: return fd_sweep_kernel<FD_INST_CPLX, MODE, R, FD_INST_PH, 3, FD_INST_EX>;
        FD_INST_ROWS(FD_INST_CASE)
#undef FD_INST_CASE
    default: return fd_sweep_kernel<FD_INST_CPLX, MODE, 0, FD_INST_PH, 3, FD_INST_EX>;
    }
}
}  // namespace

FdSweepKernelFn FD_INST_NAME(int rowd, int mode, int nn)
{
    return mode ? pick<1>(rowd, nn) : pick<0>(rowd, nn);
}
