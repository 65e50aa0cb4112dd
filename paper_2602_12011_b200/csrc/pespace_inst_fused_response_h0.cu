// fused multi-detector response kernels, class masks 1..7 (see pespace_inst.cuh)
#define PESPACE_INST_WHAT 5
#define PESPACE_INST_KIND 0
#define PESPACE_INST_HALF 0
#include "pespace_inst.cuh"
