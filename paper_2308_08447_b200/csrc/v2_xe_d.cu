#define V2_INST_STAGE 3
#define V2_INST_T double
#include "v2_inst.cuh"
