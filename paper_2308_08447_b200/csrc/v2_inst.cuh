// v2_inst.cuh -- explicit instantiation of the fast-path launchers (v2_host.cuh), one translation unit per
// (stage, precision) so that the library builds in parallel (build.py).  V2_INST_STAGE = 0 (x), 1 (y), 2 (z), 3 (x, embedded caller arrays);
// V2_INST_T = float | double.
#include "v2_host.cuh"

namespace demag {
namespace v2 {
#if V2_INST_STAGE == 0
template bool x_fwd<V2_INST_T>(int, const Ctx<V2_INST_T>&, cudaStream_t, const V2_INST_T*, CQ<V2_INST_T>*, cudaError_t*);
template bool x_fwd_sh<V2_INST_T>(int, const Ctx<V2_INST_T>&, cudaStream_t, const V2_INST_T*, cudaError_t*);
template bool x_inv<V2_INST_T>(int, const Ctx<V2_INST_T>&, cudaStream_t, const CQ<V2_INST_T>*, V2_INST_T*, cudaError_t*, int);
#elif V2_INST_STAGE == 3
template bool x_fwd_e<V2_INST_T>(int, const Ctx<V2_INST_T>&, cudaStream_t, const V2_INST_T*, CQ<V2_INST_T>*, cudaError_t*);
template bool x_inv_e<V2_INST_T>(int, const Ctx<V2_INST_T>&, cudaStream_t, const CQ<V2_INST_T>*, V2_INST_T*, cudaError_t*, int);
#elif V2_INST_STAGE == 1
template bool y_fwd<V2_INST_T>(int, const Ctx<V2_INST_T>&, cudaStream_t, int, int, const CQ<V2_INST_T>*, CQ<V2_INST_T>*, cudaError_t*);
template bool y_inv<V2_INST_T>(int, const Ctx<V2_INST_T>&, cudaStream_t, int, int, const CQ<V2_INST_T>*, CQ<V2_INST_T>*, cudaError_t*);
template bool y_inv_sh<V2_INST_T>(int, const Ctx<V2_INST_T>&, cudaStream_t, int, int, const CQ<V2_INST_T>*, cudaError_t*);
#else
template bool z_mul<V2_INST_T>(int, const Ctx<V2_INST_T>&, cudaStream_t, int, int, CQ<V2_INST_T>*, const typename kchunks<V2_INST_T>::V*, cudaError_t*);
template bool y_film<V2_INST_T>(int, const Ctx<V2_INST_T>&, cudaStream_t, CQ<V2_INST_T>*, const typename kchunks<V2_INST_T>::V*, cudaError_t*);
#endif
}  // namespace v2
}  // namespace demag
