// rflbm_step_inst.cu — explicit instantiation of the step kernels for ONE (precision, phase) pair:
// compiled six times by build.py with -DRFLBM_INST_REAL=double|float -DRFLBM_INST_PHASE=0|1|2.
#include "rflbm_host.cuh"

#if !defined(RFLBM_INST_REAL) || !defined(RFLBM_INST_PHASE)
#error "compile with -DRFLBM_INST_REAL=double|float -DRFLBM_INST_PHASE=0|1|2"
#endif

template void dispatch_variant<RFLBM_INST_REAL, RFLBM_INST_PHASE>(rflbm*, const StepParams<RFLBM_INST_REAL>&, int, bool);
