// common.cuh -- shared device/host helpers of libpaci (sm_100a only).
#pragma once

#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <cstdio>
#include <string>

#include "../../include/paci.h"

namespace paci {

// ---------------------------------------------------------------- error + launch bookkeeping
extern thread_local std::string g_last_error;
extern std::atomic<int64_t> g_launches;

int fail(int code, const char* fmt, ...);

#define PACI_CUDA_OK(expr)                                                              \
  do {                                                                                  \
    cudaError_t e__ = (expr);                                                           \
    if (e__ != cudaSuccess)                                                             \
      return ::paci::fail(PACI_ECUDA, "%s:%d %s -> %s", __FILE__, __LINE__, #expr,      \
                          cudaGetErrorString(e__));                                     \
  } while (0)

// Programmatic dependent launch (PDL).  Every kernel of the library is launched with
// cudaLaunchAttributeProgrammaticStreamSerialization and starts with PACI_PDL_SYNC (after its own on-chip set-up:
// barrier init, TMEM allocation, descriptor prefetch): `griddepcontrol.wait` blocks until the previous kernel of the
// stream has COMPLETED and its memory is visible, so no kernel touches global memory early; `launch_dependents` then
// lets the NEXT kernel of the stream be scheduled onto SMs as they free up, where it runs its set-up and parks in its
// own wait.  What is hidden is the launch latency and the prologue, never a data dependency.
#ifndef PACI_NO_PDL
#define PACI_PDL_SYNC do { asm volatile("griddepcontrol.wait;" ::: "memory"); \
                           asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); } while (0)
#define PACI_PDL_ATTR 1
#else
#define PACI_PDL_SYNC do {} while (0)
#define PACI_PDL_ATTR 0
#endif

template <typename... KArgs, typename... Args>
inline cudaError_t launch_kernel(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream,
                                 Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = PACI_PDL_ATTR;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

// every kernel launch goes through this so that paci_launch_count() is exact
#define PACI_LAUNCH(kernel, grid, block, smem, stream, ...)                             \
  do {                                                                                  \
    PACI_CUDA_OK(::paci::launch_kernel(kernel, dim3(grid), dim3(block), (smem), (stream), __VA_ARGS__)); \
    ::paci::g_launches.fetch_add(1, std::memory_order_relaxed);                         \
  } while (0)

// ---------------------------------------------------------------- dtype traits
typedef __nv_bfloat16 bf16;

template <typename T> struct Vec;                 // 16-byte vector of T
template <> struct Vec<float> { static constexpr int N = 4; };
template <> struct Vec<bf16>  { static constexpr int N = 8; };

__device__ __forceinline__ float to_f(float x) { return x; }
__device__ __forceinline__ float to_f(bf16 x) { return __bfloat162float(x); }
template <typename T> __device__ __forceinline__ T from_f(float x);
template <> __device__ __forceinline__ float from_f<float>(float x) { return x; }
template <> __device__ __forceinline__ bf16 from_f<bf16>(float x) { return __float2bfloat16_rn(x); }

// 16-byte global load / store of Vec<T>::N elements, converted to / from fp32 registers
template <typename T> __device__ __forceinline__ void load_vec(const T* p, float (&v)[Vec<T>::N]);
template <> __device__ __forceinline__ void load_vec<float>(const float* p, float (&v)[4]) {
  float4 t = *reinterpret_cast<const float4*>(p);
  v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
}
template <> __device__ __forceinline__ void load_vec<bf16>(const bf16* p, float (&v)[8]) {
  uint4 t = *reinterpret_cast<const uint4*>(p);
  const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&t);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    float2 f = __bfloat1622float2(h[i]);
    v[2 * i] = f.x; v[2 * i + 1] = f.y;
  }
}
template <typename T> __device__ __forceinline__ void store_vec(T* p, const float (&v)[Vec<T>::N]);
template <> __device__ __forceinline__ void store_vec<float>(float* p, const float (&v)[4]) {
  *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
}
template <> __device__ __forceinline__ void store_vec<bf16>(bf16* p, const float (&v)[8]) {
  uint4 t;
  __nv_bfloat162* h = reinterpret_cast<__nv_bfloat162*>(&t);
#pragma unroll
  for (int i = 0; i < 4; ++i) h[i] = __floats2bfloat162_rn(v[2 * i], v[2 * i + 1]);
  *reinterpret_cast<uint4*>(p) = t;
}
// raw 16-byte vector kept PACKED in registers (4 registers instead of Vec<T>::N) and unpacked on use
template <typename T> __device__ __forceinline__ uint4 load_raw(const T* p) { return *reinterpret_cast<const uint4*>(p); }
template <typename T> __device__ __forceinline__ void unpack_raw(const uint4& t, float (&v)[Vec<T>::N]);
template <> __device__ __forceinline__ void unpack_raw<float>(const uint4& t, float (&v)[4]) {
  v[0] = __uint_as_float(t.x); v[1] = __uint_as_float(t.y); v[2] = __uint_as_float(t.z); v[3] = __uint_as_float(t.w);
}
template <> __device__ __forceinline__ void unpack_raw<bf16>(const uint4& t, float (&v)[8]) {
  const uint32_t w[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {                 // bf16 -> fp32 is a 16-bit shift
    v[2 * i] = __uint_as_float(w[i] << 16);
    v[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
  }
}
// N consecutive fp32 values (N = 4 or 8) as float4 loads
template <int N> __device__ __forceinline__ void load_f32(const float* p, float (&v)[N]) {
#pragma unroll
  for (int i = 0; i < N / 4; ++i) {
    float4 t = reinterpret_cast<const float4*>(p)[i];
    v[4 * i] = t.x; v[4 * i + 1] = t.y; v[4 * i + 2] = t.z; v[4 * i + 3] = t.w;
  }
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// GELU (tanh form, R12) of the bf16 path: MUFU.TANH (max abs error ~5e-4, below the bf16 rounding
// of the result).  Shared by gelu_fwd_kernel and the fused MLP-up GEMM epilogue so both give the same bits.
__device__ __forceinline__ float tanh_fast(float u) {
  float r;
  asm("tanh.approx.f32 %0, %1;" : "=f"(r) : "f"(u));
  return r;
}
// gelu(p) = 0.5 p (1 + tanh(C (p + A p^3))) as five FMA-class operations and the tanh: u = p (C + C A p^2),
// h = 0.5 p, result = h + h tanh(u)
__device__ __forceinline__ float gelu_bf16(float p) {
  const float u = p * fmaf(0.7978845608028654f * 0.044715f, p * p, 0.7978845608028654f);
  const float h = 0.5f * p;
  return fmaf(h, tanh_fast(u), h);
}

static inline int ceil_div(long long a, long long b) { return (int)((a + b - 1) / b); }
static inline size_t align_up(size_t a, size_t b) { return (a + b - 1) / b * b; }

int num_sms();                                            // of the current device
// cudaFuncAttributeMaxDynamicSharedMemorySize, once per (current device, kernel); thread-safe
int set_max_dynamic_smem(const void* func, int bytes);

// ---------------------------------------------------------------- sampled kernel timing (prof.cu)
enum ProfCat { PC_GEMM_FWD = 0, PC_GEMM_DGRAD, PC_GEMM_WGRAD, PC_ATTN_FWD, PC_ATTN_BWD, PC_LN_FWD, PC_LN_BWD,
               PC_GELU_FWD, PC_GELU_BWD, PC_COLSUM, PC_EMBED, PC_SOFTMAX_CE, PC_ADAMW, PC_OTHER, PC_GEMM_BWD_PAIR };
struct ProfScope {   // counts the launch; every stride-th one is timed with events on stream s
  ProfScope(int cat, double flops, double bytes, cudaStream_t s);
  ~ProfScope();
  int idx_;
  cudaStream_t stream_;
};
void prof_set_peer_streams(const cudaStream_t* streams, int n);   // sampled launches run alone w.r.t. these
int stage_cfg_field(const ::paci_stage* st, int field);   // i-th int32 of the stage's paci_stage_config

// ---------------------------------------------------------------- kernel launchers (host)
// dtype: PACI_FP32 | PACI_BF16.  All return PACI_OK or a negative code.
int ln_fwd(int dtype, int rows, int D, const void* x, const void* res, const float* g, const float* b,
           void* xsum, void* y, float* mean, float* rstd, cudaStream_t s);
int ln_bwd(int dtype, int rows, int D, const void* dy, const void* x, const float* mean, const float* rstd,
           const float* g, const void* dres, void* dx, float* Gg, float* Gb, float* Gcol, cudaStream_t s);
int gelu_fwd(int dtype, size_t n, const void* p, void* out, cudaStream_t s);
int gelu_bwd(int dtype, int rows, int cols, const void* dg, const void* p, void* dp, float* Gbias,
             cudaStream_t s);
int colsum(int dtype, int rows, int cols, const void* x, float* G, cudaStream_t s);
// token / target ids outside [0, vocab) are clamped and raise *err (sticky device word, may be NULL)
int embed_fwd(int dtype, int mu, int T, int D, const int32_t* tok, const float* wte, const float* wpe,
              void* x, int vocab, int64_t* err, cudaStream_t s);
int embed_bwd(int dtype, int mu, int T, int D, const int32_t* tok, const void* dx, float* Gwte,
              float* Gwpe, int vocab, cudaStream_t s);
int softmax_ce(int dtype, int rows, int V, int ldz, void* z, const int32_t* tgt, float* loss, int64_t* err,
               cudaStream_t s);
// Dropout with a counter-based mask: element e of a [rows, cols] tensor is kept iff word (e % 4) of
// Philox4x32-10(counter = (e / 4 lo, e / 4 hi, mb_id lo, site), key = seed) >= floor(p 2^32); kept values are
// scaled by 1 / (1 - p).  out may alias x.  Forward and backward are the same map (the mask is regenerated).
int dropout(int dtype, size_t n, const void* x, void* out, float p, uint64_t seed, int64_t mb_id, int site,
            cudaStream_t s);
int adamw(size_t n, size_t n_decay, float* w, float* m, float* v, float* G, void* shadow, int k, int64_t t,
          float lr, float beta1, float beta2, float eps, float wd, int64_t* version_word, cudaStream_t s);
int cast_shadow(size_t n, const float* w, void* shadow, cudaStream_t s);          // bf16 shadow of fp32
int stamp_version(const int64_t* version_word, int64_t* dst, cudaStream_t s);     // *dst = *version_word
int split_tokens(int mu, int T, const int32_t* tok_tp1, int32_t* inp, int32_t* tgt, cudaStream_t s);

// GEMM: see paci_op_gemm in paci.h for layouts; lda/ldb/ldc are row strides in elements.
// gemm() dispatches on dtype.
int gemm(int dtype, int layout, int M, int N, int K, const void* A, int lda, const void* B, int ldb,
         const float* bias, void* C, int ldc, int out_f32_accum, cudaStream_t s);
int gemm_simt(int dtype, int layout, int M, int N, int K, const void* A, int lda, const void* B, int ldb,
              const float* bias, void* C, int ldc, int out_f32_accum, cudaStream_t s);
int gemm_tc(int layout, int M, int N, int K, const void* A, int lda, const void* B, int ldb, const float* bias,
            void* C, int ldc, int out_f32_accum, cudaStream_t s, void* gelu_out = nullptr);
// One GEMM as a value (same fields as gemm()'s arguments).
// Extra outputs of the out-projection dgrad's epilogue (the prologue of row a17): with C = dO [mu T, H 64] it also
// writes delta[b,h,t] = sum_d dO[b,t,h,d] O[b,t,h,d] and lse2 = lse log2(e), both fp32 [mu, H, T] -- what the separate
// attn_delta kernel computes, without re-reading dO.
struct AttnDeltaOut {
  const void* o; int ldo;            // attention output O, bf16 [mu T, H 64]
  const float* lse;                  // [mu, H, T] from the forward
  float* delta; float* lse2;         // [mu, H, T] each
  int T, H;
};
struct GemmDesc {
  int layout, M, N, K;
  const void* A; int lda;
  const void* B; int ldb;
  const float* bias;
  void* C; int ldc;
  int out_f32_accum;
  void* gelu_out;
  const AttnDeltaOut* delta;         // NULL unless this is the out-projection dgrad (bf16 only)
};
int gemm_tc_multi(const GemmDesc* d, int n, cudaStream_t s);       // n <= 2 problems in ONE persistent launch
// The backward pair of one linear layer y = x W^T: G_W += dy^T x (wgrad, beta = 1, Alg. 1 line 13) and dx = dy W
// (dgrad with the CURRENT W, Eq. 1).  bf16: ONE tcgen05 launch whose CTA pairs share both problems' k-blocks evenly;
// fp32: the two FFMA GEMMs.  dy [M, N_out] (row stride ld_dy), x [M, K_in], W [N_out, K_in], dx [M, K_in].
int gemm_backward_pair(int dtype, int M, int N_out, int K_in, const void* dy, int ld_dy, const void* x, int ld_x,
                       const void* W, int ld_w, float* G_W, int ld_g, void* dx, int ld_dx, cudaStream_t s);
// C = A B^T + bias (pre-activation, stashed for backward) and Gout = gelu(C), both [M, N] with row stride ldc:
// one launch on the tcgen05 path (GELU in the GEMM epilogue, rows a7 + a8), GEMM then gelu_fwd otherwise.
int gemm_bias_gelu(int dtype, int M, int N, int K, const void* A, int lda, const void* B, int ldb, const float* bias,
                   void* C, void* Gout, int ldc, cudaStream_t s);
void gemm_tc_last_plan(int32_t* out6);
int add_vec(int dtype, size_t n, const void* a, const void* b, void* out, cudaStream_t s);  // out = a (+ b)

int attention_fwd(int dtype, int mu, int T, int H, int dh, const void* qkv, void* o, float* lse,
                  cudaStream_t s);
int attention_bwd(int dtype, int mu, int T, int H, int dh, const void* dout, const void* qkv, const void* o,
                  const float* lse, void* dqkv, float* scratch, float* Gbias, cudaStream_t s, int scratch_prepared = 0);
int out_proj_backward(int dtype, int mu, int T, int H, int dh, const void* dy, const void* o, const void* Wo,
                      float* G_Wo, void* d_o, const float* lse, float* attn_scratch, int* prepared, cudaStream_t s);
size_t attention_bwd_scratch_bytes(int dtype, int mu, int T, int H, int dh);
int attention_fwd_simt(int dtype, int mu, int T, int H, int dh, const void* qkv, void* o, float* lse,
                       cudaStream_t s);
int attention_bwd_simt(int dtype, int mu, int T, int H, int dh, const void* dout, const void* qkv,
                       const void* o, const float* lse, void* dqkv, float* scratch, cudaStream_t s);

}  // namespace paci
