// encode_tensor.cu -- tcgen05/TMEM segment encode (kernel family HYPIC_IMPL_TENSOR).  Placeholder: the
// family reports "not supported" until the chunked kernel lands, so AUTO falls through to the SIMT family.
#include "common.cuh"

namespace hypic {
bool encode_tensor_shape_ok(int32_t, int32_t, int32_t, int, int) { return false; }
size_t encode_tensor_workspace(int32_t, int32_t, int32_t, int32_t, int32_t, int, int) { return 0; }
int encode_tensor(const EncodeArgs&) { return HYPIC_ERR_UNSUPPORTED; }
}  // namespace hypic
