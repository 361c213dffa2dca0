// placeholder until the tcgen05 kernel lands (next commit)
#include "common.cuh"
namespace paci {
int gemm_tc(int, int, int, int, const void*, int, const void*, int, const float*, void*, int, int, cudaStream_t) {
  return fail(PACI_EINVAL, "tcgen05 GEMM not built yet; set PACI_GEMM=simt");
}
}
