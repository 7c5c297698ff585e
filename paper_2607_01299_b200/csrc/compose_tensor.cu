// compose_tensor.cu -- tcgen05/TMEM composition (kernel family HYPIC_IMPL_TENSOR).  Placeholder: the family
// reports "not supported" until the 3xTF32 kernel lands, so AUTO falls through to the SIMT family.
#include "common.cuh"

namespace hypic {
bool compose_tensor_shape_ok(int32_t, int32_t, int32_t) { return false; }
int compose_tensor(const ComposeArgs&) { return HYPIC_ERR_UNSUPPORTED; }
}  // namespace hypic
