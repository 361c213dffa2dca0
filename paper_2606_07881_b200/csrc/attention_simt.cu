// attention_simt.cu -- direct (non-tiled) causal attention forward/backward on CUDA cores.
// Product path in PACI_FP32 mode (tiny config, any head dim <= 128, 1e-5 parity); in PACI_BF16 mode
// it is only a debugging aid behind PACI_ATTN=simt.  Rows a4 / a17 of SURVEY.md 8(a).
//
// qkv is packed [mu, T, 3D] with q | k | v in the last axis and head h at columns h*dh..(h+1)*dh-1
// (R17).  Backward recomputes the probabilities from the stashed q, k and lse (no
// parameter involved, so this is not the checkpointed variant of P:282).
#include "common.cuh"

namespace paci {

template <typename T> __device__ __forceinline__ float exp_acc(float x);
template <> __device__ __forceinline__ float exp_acc<float>(float x) { return expf(x); }
template <> __device__ __forceinline__ float exp_acc<bf16>(float x) { return __expf(x); }

__device__ __forceinline__ float block_reduce(float v, bool is_max, float* red) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  v = is_max ? warp_max(v) : warp_sum(v);
  __syncthreads();
  if (lane == 0) red[w] = v;
  __syncthreads();
  float r = is_max ? -INFINITY : 0.f;
  for (int i = 0; i < nw; ++i) r = is_max ? fmaxf(r, red[i]) : r + red[i];
  return r;
}

template <typename T>
__global__ void __launch_bounds__(128) attn_fwd_simt_kernel(int T_, int H, int dh, const T* __restrict__ qkv,
                                                            T* __restrict__ o, float* __restrict__ lse) {
  PACI_PDL_SYNC;
  extern __shared__ float sm[];     // q[dh] | s[T]
  __shared__ float red[4];
  float* q = sm;
  float* sc = sm + dh;
  const int i = blockIdx.x, h = blockIdx.y, b = blockIdx.z;
  const int D = H * dh;
  const float scale = rsqrtf((float)dh);
  const T* base = qkv + (size_t)b * T_ * 3 * D;
  for (int d = threadIdx.x; d < dh; d += blockDim.x) q[d] = to_f(base[(size_t)i * 3 * D + h * dh + d]);
  __syncthreads();
  float mx = -INFINITY;
  for (int j = threadIdx.x; j <= i; j += blockDim.x) {
    const T* kj = base + (size_t)j * 3 * D + D + h * dh;
    float s = 0.f;
    for (int d = 0; d < dh; ++d) s = fmaf(q[d], to_f(kj[d]), s);
    s *= scale;
    sc[j] = s;
    mx = fmaxf(mx, s);
  }
  mx = block_reduce(mx, true, red);
  float sum = 0.f;
  for (int j = threadIdx.x; j <= i; j += blockDim.x) {
    const float p = exp_acc<T>(sc[j] - mx);
    sc[j] = p;
    sum += p;
  }
  sum = block_reduce(sum, false, red);
  if (threadIdx.x == 0) lse[((size_t)b * H + h) * T_ + i] = mx + logf(sum);
  const float inv = 1.f / sum;
  for (int d = threadIdx.x; d < dh; d += blockDim.x) {
    float acc = 0.f;
    for (int j = 0; j <= i; ++j) acc = fmaf(sc[j], to_f(base[(size_t)j * 3 * D + 2 * D + h * dh + d]), acc);
    o[((size_t)b * T_ + i) * D + h * dh + d] = from_f<T>(acc * inv);
  }
}

// dq_i and delta_i = sum_d do_i[d] * o_i[d]
template <typename T>
__global__ void __launch_bounds__(128) attn_bwd_dq_simt_kernel(int T_, int H, int dh, const T* __restrict__ dout,
                                                               const T* __restrict__ qkv, const T* __restrict__ o,
                                                               const float* __restrict__ lse, T* __restrict__ dqkv,
                                                               float* __restrict__ delta) {
  PACI_PDL_SYNC;
  extern __shared__ float sm[];     // q[dh] | do[dh] | ds[T]
  __shared__ float red[4];
  float* q = sm;
  float* dO = sm + dh;
  float* ds = sm + 2 * dh;
  const int i = blockIdx.x, h = blockIdx.y, b = blockIdx.z;
  const int D = H * dh;
  const float scale = rsqrtf((float)dh);
  const T* base = qkv + (size_t)b * T_ * 3 * D;
  float part = 0.f;
  for (int d = threadIdx.x; d < dh; d += blockDim.x) {
    q[d] = to_f(base[(size_t)i * 3 * D + h * dh + d]);
    const size_t oi = ((size_t)b * T_ + i) * D + h * dh + d;
    dO[d] = to_f(dout[oi]);
    part += dO[d] * to_f(o[oi]);
  }
  const float dl = block_reduce(part, false, red);
  const float L = lse[((size_t)b * H + h) * T_ + i];
  if (threadIdx.x == 0) delta[((size_t)b * H + h) * T_ + i] = dl;
  __syncthreads();
  for (int j = threadIdx.x; j <= i; j += blockDim.x) {
    const T* kj = base + (size_t)j * 3 * D + D + h * dh;
    const T* vj = base + (size_t)j * 3 * D + 2 * D + h * dh;
    float s = 0.f, dp = 0.f;
    for (int d = 0; d < dh; ++d) {
      s = fmaf(q[d], to_f(kj[d]), s);
      dp = fmaf(dO[d], to_f(vj[d]), dp);
    }
    ds[j] = exp_acc<T>(s * scale - L) * (dp - dl);
  }
  __syncthreads();
  for (int d = threadIdx.x; d < dh; d += blockDim.x) {
    float acc = 0.f;
    for (int j = 0; j <= i; ++j) acc = fmaf(ds[j], to_f(base[(size_t)j * 3 * D + D + h * dh + d]), acc);
    dqkv[((size_t)b * T_ + i) * 3 * D + h * dh + d] = from_f<T>(acc * scale);
  }
}

// dk_j = scale * sum_{i>=j} ds_ij q_i ;  dv_j = sum_{i>=j} P_ij do_i
template <typename T>
__global__ void __launch_bounds__(128) attn_bwd_dkv_simt_kernel(int T_, int H, int dh, const T* __restrict__ dout,
                                                                const T* __restrict__ qkv,
                                                                const float* __restrict__ lse,
                                                                const float* __restrict__ delta,
                                                                T* __restrict__ dqkv) {
  PACI_PDL_SYNC;
  extern __shared__ float sm[];     // k[dh] | v[dh] | P[T] | ds[T]
  float* k = sm;
  float* v = sm + dh;
  float* P = sm + 2 * dh;
  float* ds = P + T_;
  const int j = blockIdx.x, h = blockIdx.y, b = blockIdx.z;
  const int D = H * dh;
  const float scale = rsqrtf((float)dh);
  const T* base = qkv + (size_t)b * T_ * 3 * D;
  for (int d = threadIdx.x; d < dh; d += blockDim.x) {
    k[d] = to_f(base[(size_t)j * 3 * D + D + h * dh + d]);
    v[d] = to_f(base[(size_t)j * 3 * D + 2 * D + h * dh + d]);
  }
  __syncthreads();
  for (int i = j + threadIdx.x; i < T_; i += blockDim.x) {
    const T* qi = base + (size_t)i * 3 * D + h * dh;
    const T* doi = dout + ((size_t)b * T_ + i) * D + h * dh;
    float s = 0.f, dp = 0.f;
    for (int d = 0; d < dh; ++d) {
      s = fmaf(to_f(qi[d]), k[d], s);
      dp = fmaf(to_f(doi[d]), v[d], dp);
    }
    const size_t li = ((size_t)b * H + h) * T_ + i;
    const float p = exp_acc<T>(s * scale - lse[li]);
    P[i] = p;
    ds[i] = p * (dp - delta[li]);
  }
  __syncthreads();
  for (int d = threadIdx.x; d < dh; d += blockDim.x) {
    float ak = 0.f, av = 0.f;
    for (int i = j; i < T_; ++i) {
      ak = fmaf(ds[i], to_f(base[(size_t)i * 3 * D + h * dh + d]), ak);
      av = fmaf(P[i], to_f(dout[((size_t)b * T_ + i) * D + h * dh + d]), av);
    }
    dqkv[((size_t)b * T_ + j) * 3 * D + D + h * dh + d] = from_f<T>(ak * scale);
    dqkv[((size_t)b * T_ + j) * 3 * D + 2 * D + h * dh + d] = from_f<T>(av);
  }
}

int attention_fwd_simt(int dtype, int mu, int T_, int H, int dh, const void* qkv, void* o, float* lse,
                       cudaStream_t s) {
  dim3 grid(T_, H, mu);
  const size_t smem = (size_t)(dh + T_) * sizeof(float);
  if (smem > 48 * 1024) return fail(PACI_EINVAL, "attention_simt: T=%d too long for the direct kernel", T_);
  if (dtype == PACI_BF16)
    PACI_LAUNCH(attn_fwd_simt_kernel<bf16>, grid, 128, smem, s, T_, H, dh, (const bf16*)qkv, (bf16*)o, lse);
  else
    PACI_LAUNCH(attn_fwd_simt_kernel<float>, grid, 128, smem, s, T_, H, dh, (const float*)qkv, (float*)o, lse);
  return PACI_OK;
}

int attention_bwd_simt(int dtype, int mu, int T_, int H, int dh, const void* dout, const void* qkv, const void* o,
                       const float* lse, void* dqkv, float* scratch, cudaStream_t s) {
  dim3 grid(T_, H, mu);
  const size_t smem1 = (size_t)(2 * dh + T_) * sizeof(float), smem2 = (size_t)(2 * dh + 2 * T_) * sizeof(float);
  if (smem2 > 48 * 1024) return fail(PACI_EINVAL, "attention_simt: T=%d too long for the direct kernel", T_);
  float* delta = scratch;
  if (dtype == PACI_BF16) {
    PACI_LAUNCH(attn_bwd_dq_simt_kernel<bf16>, grid, 128, smem1, s, T_, H, dh, (const bf16*)dout, (const bf16*)qkv,
                (const bf16*)o, lse, (bf16*)dqkv, delta);
    PACI_LAUNCH(attn_bwd_dkv_simt_kernel<bf16>, grid, 128, smem2, s, T_, H, dh, (const bf16*)dout,
                (const bf16*)qkv, lse, delta, (bf16*)dqkv);
  } else {
    PACI_LAUNCH(attn_bwd_dq_simt_kernel<float>, grid, 128, smem1, s, T_, H, dh, (const float*)dout,
                (const float*)qkv, (const float*)o, lse, (float*)dqkv, delta);
    PACI_LAUNCH(attn_bwd_dkv_simt_kernel<float>, grid, 128, smem2, s, T_, H, dh, (const float*)dout,
                (const float*)qkv, lse, delta, (float*)dqkv);
  }
  return PACI_OK;
}

}  // namespace paci
