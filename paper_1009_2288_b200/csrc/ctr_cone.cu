// 3D circular cone-beam projector pair (placeholder until the 3D kernels land).
#include "ctr_common.cuh"
#include "ctr_internal.h"

namespace ctr {
int cone_build_tables(ctr_handle* h) { return set_err(h, CTR_EINVAL, "3D cone beam is not implemented yet"); }
int cone_forward(ctr_handle* h, const float*, float*, int, const float*, cudaStream_t) { return set_err(h, CTR_EINVAL, "3D"); }
int cone_back(ctr_handle* h, const float*, float*, int, const float*, float*, cudaStream_t) { return set_err(h, CTR_EINVAL, "3D"); }
}  // namespace ctr
