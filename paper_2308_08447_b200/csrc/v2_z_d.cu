#define V2_INST_STAGE 2
#define V2_INST_T double
#include "v2_inst.cuh"
