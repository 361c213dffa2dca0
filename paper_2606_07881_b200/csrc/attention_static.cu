// attention_static.cu -- paci_op_attention_bwd_static: attention backward for callers that
// may not allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// The existing entry point, paci_op_attention_bwd, takes its scratch (delta = rowsum(dO * O), lse * log2(e) and the two
// work counters of the persistent tcgen05 kernels; fp32: delta only) from the caller.  Here the scratch is ONE
// file-scope device array of PACI_ATTENTION_BWD_STATIC_MAX_BYTES: every GPU that loads the library holds it until the
// process exits.  Nothing else differs: the same kernels run, through the same dispatch (attention_bwd in ops.cu).
//
// In HOST code the array's name is a host-side stand-in, not a device address (a kernel given it would fault or use the
// wrong memory), so the device address is looked up with cudaGetSymbolAddress -- once per device, with that device
// current, under a mutex -- and that pointer is what the kernels receive.
//
// Every call on a device shares the array.  It keeps the last call's contents; that is harmless because each call
// rewrites all of what it reads before reading it, in stream order: the delta pass (first launch) writes delta, lse2
// and zeroes both work counters.  Two calls that OVERLAP on the GPU (different streams, or graph branches without an
// edge between them) race on the array and on the counters: serialise them.
//
// No cudaMalloc / cudaFree / allocating library routine is reached from here: tensor maps are encoded on the host stack
// (cuTensorMapEncodeTiled), cudaFuncSetAttribute and the launches allocate nothing.  (With paci_profile_begin active,
// the sampling profiler creates CUDA events: do not profile inside a capture.)
#include <mutex>

#include "common.cuh"

namespace paci {
namespace {

static __device__ __align__(256) unsigned char g_attn_bwd_scratch[PACI_ATTENTION_BWD_STATIC_MAX_BYTES];

constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
float* g_scratch_addr[MAX_DEVICES] = {};      // device address of g_attn_bwd_scratch on device i (nullptr: not looked up)

// set-up, once per device, with that device current
int static_scratch(float** out) {
  int dev = -1;
  PACI_CUDA_OK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= MAX_DEVICES) return fail(PACI_EINVAL, "paci_op_attention_bwd_static: device %d out of range", dev);
  std::lock_guard<std::mutex> g(g_mu);
  if (g_scratch_addr[dev] == nullptr) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_attn_bwd_scratch);
    if (e != cudaSuccess || p == nullptr)
      return fail(PACI_ECUDA, "paci_op_attention_bwd_static: cudaGetSymbolAddress on device %d -> %s", dev,
                  cudaGetErrorString(e));
    g_scratch_addr[dev] = static_cast<float*>(p);
  }
  *out = g_scratch_addr[dev];
  return PACI_OK;
}

}  // namespace
}  // namespace paci

using namespace paci;

extern "C" int paci_op_attention_bwd_static(int dtype, int mu, int T, int H, int dh, const void* dout, const void* qkv,
                                            const void* o, const float* lse, void* dqkv, void* stream) {
  if (mu <= 0 || T <= 0 || H <= 0 || dh <= 0)
    return fail(PACI_EINVAL, "paci_op_attention_bwd_static: mu, T, H, dh must be positive");
  if (dout == nullptr || qkv == nullptr || o == nullptr || lse == nullptr || dqkv == nullptr)
    return fail(PACI_EINVAL, "paci_op_attention_bwd_static: NULL input or output");
  // the size test comes before any CUDA call: a shape beyond the fixed array is refused, never truncated
  const size_t need = attention_bwd_scratch_bytes(dtype, mu, T, H, dh);
  if (need > (size_t)PACI_ATTENTION_BWD_STATIC_MAX_BYTES)
    return fail(PACI_EINVAL,
                "paci_op_attention_bwd_static: mu=%d T=%d H=%d needs %zu bytes of scratch, the static array holds %zu "
                "(mu*H*T <= %zu); use paci_op_attention_bwd with caller-provided scratch",
                mu, T, H, need, (size_t)PACI_ATTENTION_BWD_STATIC_MAX_BYTES,
                ((size_t)PACI_ATTENTION_BWD_STATIC_MAX_BYTES - 64) / 8);
  float* scratch = nullptr;
  const int rc = static_scratch(&scratch);
  if (rc != PACI_OK) return rc;
  return attention_bwd(dtype, mu, T, H, dh, dout, qkv, o, lse, dqkv, scratch, nullptr, (cudaStream_t)stream, 0);
}
