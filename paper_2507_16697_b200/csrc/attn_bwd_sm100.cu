// attn_bwd_sm100.cu -- placeholder until the tcgen05 backward lands (reports "not supported").
#include "kernels.cuh"
namespace ringx {
cudaError_t launch_attn_chunk_bwd_sm100(const void*, const void*, const void*, const void*, const float*, const float*,
                                        float*, void*, void*, int, int, int, int, int, float, cudaStream_t) {
  return cudaErrorNotSupported;
}
}  // namespace ringx
