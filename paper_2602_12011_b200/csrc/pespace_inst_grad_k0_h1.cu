// adjoint-gradient kernels, detector kind 0, class masks 8..15 (see pespace_inst.cuh)
#define PESPACE_INST_WHAT 3
#define PESPACE_INST_KIND 0
#define PESPACE_INST_HALF 1
#include "pespace_inst.cuh"
