#define V2_INST_STAGE 2
#define V2_INST_T float
#include "v2_inst.cuh"
