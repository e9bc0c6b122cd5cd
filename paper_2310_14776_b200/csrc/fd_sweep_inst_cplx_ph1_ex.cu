// Instantiations of the sweep kernel: complex128, PH = 1, with the expectation-value epilogue (one translation unit of several: see build.py and
// fd_sweep_inst.h).
#define FD_INST_CPLX true
#define FD_INST_PH 1
#define FD_INST_EX true
#define FD_INST_NAME fd_sweep_pick_cplx_ph1_ex
#define FD_INST_ROWS(X) X(48) X(96) X(144) X(192)
#include "fd_sweep_inst.h"
