// attn_tc.cu — tcgen05 flash attention (placeholder until the tensor-core kernel lands).
#include "common.cuh"
namespace dit {
bool attn_tc_supported(const AttnArgs&) { return false; }
dit_status launch_attn_tc(const AttnArgs&, cudaStream_t) {
  set_error("tcgen05 attention not built");
  return DIT_ERR_UNSUPPORTED;
}
}  // namespace dit
