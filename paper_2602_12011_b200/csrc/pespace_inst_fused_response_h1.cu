// fused multi-detector response kernels, class masks 8..15 (see pespace_inst.cuh)
#define PESPACE_INST_WHAT 5
#define PESPACE_INST_KIND 0
#define PESPACE_INST_HALF 1
#include "pespace_inst.cuh"
