// fused multi-detector likelihood kernels, class masks 1..7 (see pespace_inst.cuh)
#define PESPACE_INST_WHAT 4
#define PESPACE_INST_KIND 0
#define PESPACE_INST_HALF 0
#include "pespace_inst.cuh"
