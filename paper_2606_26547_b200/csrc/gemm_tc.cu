// gemm_tc.cu -- placeholder until the tcgen05 kernel lands: reports "not supported" so callers use
// the CUDA-core contraction.
#include "common.cuh"
namespace hdc {
struct TcContext { int dummy; };
TcContext* tc_context_create() { return nullptr; }
void tc_context_destroy(TcContext*) {}
cudaError_t launch_gemm_tc(TcContext*, const void*, const void*, int, int64_t, int, int, int64_t, int64_t,
                           const Epilogue&, int, cudaStream_t, int64_t*) {
  return cudaErrorNotSupported;
}
}  // namespace hdc
