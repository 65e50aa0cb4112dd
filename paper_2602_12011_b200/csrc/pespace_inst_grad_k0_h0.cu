// adjoint-gradient kernels, detector kind 0, class masks 1..7 (see pespace_inst.cuh)
#define PESPACE_INST_WHAT 3
#define PESPACE_INST_KIND 0
#define PESPACE_INST_HALF 0
#include "pespace_inst.cuh"
