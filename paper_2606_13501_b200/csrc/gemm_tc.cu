// gemm_tc.cu — tcgen05 / TMEM / TMA GEMM (placeholder until the tensor-core kernel lands: reports unsupported so
// the dispatcher uses the FFMA kernel).
#include "common.cuh"
namespace dit {
bool gemm_tc_supported(int, const void*, int64_t, const void*, void*, int64_t, int, int, int) { return false; }
dit_status launch_gemm_tc(int, const void*, int64_t, const void*, const void*, void*, int64_t, int, int, int, cudaStream_t) {
  set_error("tcgen05 GEMM not built");
  return DIT_ERR_UNSUPPORTED;
}
}  // namespace dit
