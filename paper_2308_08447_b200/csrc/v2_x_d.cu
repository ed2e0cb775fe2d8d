#define V2_INST_STAGE 0
#define V2_INST_T double
#include "v2_inst.cuh"
