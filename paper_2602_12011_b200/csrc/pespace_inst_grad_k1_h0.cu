// adjoint-gradient kernels, detector kind 1, class masks 1..7 (see pespace_inst.cuh)
#define PESPACE_INST_WHAT 3
#define PESPACE_INST_KIND 1
#define PESPACE_INST_HALF 0
#include "pespace_inst.cuh"
