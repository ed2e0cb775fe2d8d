#define V2_INST_STAGE 0
#define V2_INST_T float
#include "v2_inst.cuh"
