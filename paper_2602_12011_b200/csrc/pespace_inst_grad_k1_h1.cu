// adjoint-gradient kernels, detector kind 1, class masks 8..15 (see pespace_inst.cuh)
#define PESPACE_INST_WHAT 3
#define PESPACE_INST_KIND 1
#define PESPACE_INST_HALF 1
#include "pespace_inst.cuh"
