// fused multi-detector likelihood kernels, class masks 8..15 (see pespace_inst.cuh)
#define PESPACE_INST_WHAT 4
#define PESPACE_INST_KIND 0
#define PESPACE_INST_HALF 1
#include "pespace_inst.cuh"
