// Instantiations of the sweep kernel: float64 (one translation unit of several: see build.py and
// fd_sweep_inst.h).
#define FD_INST_CPLX false
#define FD_INST_PH 0
#define FD_INST_EX false
#define FD_INST_NAME fd_sweep_pick_real
#define FD_INST_ROWS(X) X(24) X(48) X(64) X(96) X(128) X(192)
#include "fd_sweep_inst.h"
