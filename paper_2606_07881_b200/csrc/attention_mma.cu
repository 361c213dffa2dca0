// placeholder until the tensor-core attention lands (next commit)
#include "common.cuh"
namespace paci {
int attention_fwd_mma(int, int, int, const void*, void*, float*, cudaStream_t) {
  return fail(PACI_EINVAL, "tensor-core attention not built yet; set PACI_ATTN=simt");
}
int attention_bwd_mma(int, int, int, const void*, const void*, const void*, const float*, void*, float*, cudaStream_t) {
  return fail(PACI_EINVAL, "tensor-core attention not built yet; set PACI_ATTN=simt");
}
size_t attention_bwd_mma_scratch_bytes(int mu, int T, int H) { return (size_t)mu * H * T * 4; }
}
