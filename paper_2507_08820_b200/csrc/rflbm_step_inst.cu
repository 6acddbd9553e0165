// rflbm_step_inst.cu — explicit instantiation of the step kernels for ONE (precision, phase, tile width) triple:
// compiled 24 times by build.py with -DRFLBM_INST_REAL=double|float -DRFLBM_INST_PHASE=0|1|2
// -DRFLBM_INST_TX=0|32|64|128 (0 = the plain one-thread-per-site kernel).
#include "rflbm_host.cuh"

#if !defined(RFLBM_INST_REAL) || !defined(RFLBM_INST_PHASE) || !defined(RFLBM_INST_TX)
#error "compile with -DRFLBM_INST_REAL=double|float -DRFLBM_INST_PHASE=0|1|2 -DRFLBM_INST_TX=0|32|64|128"
#endif

template void dispatch_variant<RFLBM_INST_REAL, RFLBM_INST_PHASE, RFLBM_INST_TX>(rflbm*, const StepParams<RFLBM_INST_REAL>&, int);
