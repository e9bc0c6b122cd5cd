// Instantiations of the sweep kernel: complex128, Bloch-phase code PH = 0 (bit 0: x/y wraps, bit 1: z wraps) (one translation unit of several: see build.py and
// fd_sweep_inst.h).
#define FD_INST_CPLX true
#define FD_INST_PH 0
#define FD_INST_EX false
#define FD_INST_NAME fd_sweep_pick_cplx_ph0
#define FD_INST_ROWS(X) X(48) X(96) X(144) X(192)
#include "fd_sweep_inst.h"
