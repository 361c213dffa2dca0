// elementwise.cu -- the HBM-bound kernels of the PACI stage step (SURVEY.md 8(a) rows a1, a2, a6, a8,
// a11, a15, a16, a18, a19, a20).  All use 16-byte vector accesses, fp32 statistics and warp-shuffle
// reductions; grids are sized from the SM count.
#include <cmath>
#include <cstdarg>
#include <cstdlib>
#include <mutex>
#include <set>
#include <string>
#include <utility>

#include "common.cuh"
#include "tc_ptx.cuh"

namespace paci {

thread_local std::string g_last_error;
std::atomic<int64_t> g_launches{0};

int fail(int code, const char* fmt, ...) {
  char buf[1024];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_last_error = buf;
  return code;
}

// Per-device state: the SM count and the "dynamic shared memory limit raised" flags are properties of a
// (device, kernel) pair, so both are keyed by the CURRENT device, never cached process-wide.
static constexpr int MAX_DEVICES = 64;

int num_sms() {
  static std::atomic<int> n[MAX_DEVICES];
  int dev = 0;
  cudaGetDevice(&dev);
  if (dev < 0 || dev >= MAX_DEVICES) dev = 0;
  int v = n[dev].load(std::memory_order_relaxed);
  if (v == 0) {
    cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev);
    if (v <= 0) v = 148;
    n[dev].store(v, std::memory_order_relaxed);
  }
  return v;
}

int set_max_dynamic_smem(const void* func, int bytes) {
  static std::mutex mu;
  static std::set<std::pair<int, const void*>> done;
  int dev = 0;
  PACI_CUDA_OK(cudaGetDevice(&dev));
  std::lock_guard<std::mutex> g(mu);
  if (done.count({dev, func})) return PACI_OK;
  PACI_CUDA_OK(cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  done.insert({dev, func});
  return PACI_OK;
}

__device__ __forceinline__ void red_add_v4(float* dst, float a, float b, float c, float d) {
  asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

static constexpr float LN_EPS = 1e-5f;              // DESIGN.md R13
static constexpr float GELU_C = 0.7978845608028654f;  // sqrt(2/pi), R12
static constexpr float GELU_A = 0.044715f;

// =========================================================================== LayerNorm forward
// One warp per row; the row lives in registers (NV 16-byte vectors per lane).  Optionally adds a
// residual first and writes the sum (the new residual stream) -- rows a2/a6: "LN (+ residual fused)".
template <typename T, int NV>
__global__ void __launch_bounds__(256) ln_fwd_kernel(int rows, int D, const T* __restrict__ x,
                                                     const T* __restrict__ res, const float* __restrict__ g,
                                                     const float* __restrict__ b, T* __restrict__ xsum,
                                                     T* __restrict__ y, float* __restrict__ mean_out,
                                                     float* __restrict__ rstd_out) {
  PACI_PDL_SYNC;
  constexpr int V = Vec<T>::N;
  const int lane = threadIdx.x & 31;
  const int row = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (row >= rows) return;
  const int nvec = D / V;
  const size_t base = (size_t)row * D;
  float v[NV][V];
  float sum = 0.f;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    const int c = lane + 32 * i;
    if (c < nvec) {
      load_vec<T>(x + base + (size_t)c * V, v[i]);
      if (res != nullptr) {
        float r[V];
        load_vec<T>(res + base + (size_t)c * V, r);
#pragma unroll
        for (int j = 0; j < V; ++j) v[i][j] += r[j];
      }
      if (xsum != nullptr) {
        store_vec<T>(xsum + base + (size_t)c * V, v[i]);
        if (sizeof(T) == 2) {  // statistics must see the ROUNDED stream that backward will re-read
#pragma unroll
          for (int j = 0; j < V; ++j) v[i][j] = to_f(from_f<T>(v[i][j]));
        }
      }
#pragma unroll
      for (int j = 0; j < V; ++j) sum += v[i][j];
    }
  }
  const float mean = warp_sum(sum) / (float)D;
  float sq = 0.f;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    if (lane + 32 * i < nvec) {
#pragma unroll
      for (int j = 0; j < V; ++j) {
        const float d = v[i][j] - mean;
        sq += d * d;
      }
    }
  }
  const float rstd = rsqrtf(warp_sum(sq) / (float)D + LN_EPS);
  if (lane == 0) {
    mean_out[row] = mean;
    rstd_out[row] = rstd;
  }
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    const int c = lane + 32 * i;
    if (c < nvec) {
      float gg[V], bb[V], o[V];
      load_f32<V>(g + (size_t)c * V, gg);
      load_f32<V>(b + (size_t)c * V, bb);
#pragma unroll
      for (int j = 0; j < V; ++j) o[j] = (v[i][j] - mean) * rstd * gg[j] + bb[j];
      store_vec<T>(y + base + (size_t)c * V, o);
    }
  }
}

// Pipelined forward for the stage's shape (bf16, D = 1024): one block per SM; a producer thread streams 4-row groups
// of x (and the residual) into a 12-stage shared-memory ring with bulk async copies, 3 sets of 4 compute warps take
// alternate groups, one warp per row as above; gamma / beta stay in registers.  The one-wave kernel above issues
// every load, then every store (15.5 us under ncu); here loads, arithmetic and stores of different groups overlap.
constexpr int LNQ_R = 4;
template <typename T, int S, int SETS>
__global__ void __launch_bounds__((SETS * LNQ_R + 1) * 32, 1) ln_fwd_pipe_kernel(int rows, const T* __restrict__ x,
                                                                                const T* __restrict__ res,
                                                                                const float* __restrict__ g,
                                                                                const float* __restrict__ b,
                                                                                T* __restrict__ xsum, T* __restrict__ y,
                                                                                float* __restrict__ mean_out,
                                                                                float* __restrict__ rstd_out) {
  PACI_PDL_SYNC;
  constexpr int V = Vec<T>::N, NV = 4, D = NV * 32 * V;
  constexpr uint32_t RB = D * sizeof(T), TB = LNQ_R * RB, STAGE = 2 * TB;
  extern __shared__ __align__(128) uint8_t lnq_smem[];
  uint64_t* full = reinterpret_cast<uint64_t*>(lnq_smem + S * STAGE);
  uint64_t* empty = full + S;
  const int lane = threadIdx.x & 31, w = (threadIdx.x >> 5) % LNQ_R, set = (threadIdx.x >> 5) / LNQ_R;
  const int groups = rows / LNQ_R;
  if (threadIdx.x == 0) {
    for (int i = 0; i < S; ++i) {
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(&full[i])), "r"(1));
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(&empty[i])), "r"(LNQ_R));
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  auto wait = [](uint64_t* bar, uint32_t parity) { tc::mbar_wait_many(bar, parity, 41); };
  if (set == SETS) {                                      // producer
    if (lane == 0) {
      uint32_t it = 0;
      for (int gi = blockIdx.x; gi < groups; gi += gridDim.x, ++it) {
        const uint32_t st = it % S;
        wait(&empty[st], ((it / S) & 1u) ^ 1u);
        uint8_t* base = lnq_smem + st * STAGE;
        const size_t off = (size_t)gi * LNQ_R * D;
        const uint32_t fb = (uint32_t)__cvta_generic_to_shared(&full[st]);
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(fb), "r"((res != nullptr ? 2u : 1u) * TB) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"((uint32_t)__cvta_generic_to_shared(base)), "l"(x + off), "r"(TB), "r"(fb) : "memory");
        if (res != nullptr)
          asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                       ::"r"((uint32_t)__cvta_generic_to_shared(base + TB)), "l"(res + off), "r"(TB), "r"(fb) : "memory");
      }
    }
    return;
  }
  float gg[NV][V], bb[NV][V];
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    load_f32<V>(g + (size_t)(lane + 32 * i) * V, gg[i]);
    load_f32<V>(b + (size_t)(lane + 32 * i) * V, bb[i]);
  }
  uint32_t it = set;
  for (int gi = blockIdx.x + set * gridDim.x; gi < groups; gi += SETS * gridDim.x, it += SETS) {
    const uint32_t st = it % S;
    const int row = gi * LNQ_R + w;
    const size_t base = (size_t)row * D;
    wait(&full[st], (it / S) & 1u);
    const uint8_t* sx = lnq_smem + st * STAGE + w * RB;
    uint4 rx[NV], rr[NV];
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      rx[i] = *reinterpret_cast<const uint4*>(sx + (lane + 32 * i) * 16);
      if (res != nullptr) rr[i] = *reinterpret_cast<const uint4*>(sx + TB + (lane + 32 * i) * 16);
    }
    __syncwarp();
    if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"((uint32_t)__cvta_generic_to_shared(&empty[st])) : "memory");
    float v[NV][V];
    float sum = 0.f;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      unpack_raw<T>(rx[i], v[i]);
      if (res != nullptr) {
        float r[V];
        unpack_raw<T>(rr[i], r);
#pragma unroll
        for (int j = 0; j < V; ++j) v[i][j] += r[j];
      }
      if (xsum != nullptr) {
        store_vec<T>(xsum + base + (size_t)(lane + 32 * i) * V, v[i]);
#pragma unroll
        for (int j = 0; j < V; ++j) v[i][j] = to_f(from_f<T>(v[i][j]));   // statistics see the ROUNDED stream
      }
#pragma unroll
      for (int j = 0; j < V; ++j) sum += v[i][j];
    }
    const float mean = warp_sum(sum) / (float)D;
    float sq = 0.f;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
#pragma unroll
      for (int j = 0; j < V; ++j) {
        const float d = v[i][j] - mean;
        sq += d * d;
      }
    }
    const float rstd = rsqrtf(warp_sum(sq) / (float)D + LN_EPS);
    if (lane == 0) {
      mean_out[row] = mean;
      rstd_out[row] = rstd;
    }
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      float o[V];
#pragma unroll
      for (int j = 0; j < V; ++j) o[j] = (v[i][j] - mean) * rstd * gg[i][j] + bb[i][j];
      store_vec<T>(y + base + (size_t)(lane + 32 * i) * V, o);
    }
  }
}

template <typename T>
static int ln_fwd_t(int rows, int D, const void* x, const void* res, const float* g, const float* b,
                    void* xsum, void* y, float* mean, float* rstd, cudaStream_t s) {
  constexpr int V = Vec<T>::N;
  if (D % V != 0) return fail(PACI_EINVAL, "layernorm: D=%d not a multiple of %d", D, V);
  if constexpr (sizeof(T) == 2) {
    if (D == 1024 && rows % LNQ_R == 0 && (uintptr_t)x % 16 == 0 && (uintptr_t)res % 16 == 0) {
      constexpr int S = 12, SETS = 3;
      auto kern = ln_fwd_pipe_kernel<T, S, SETS>;
      const uint32_t smem = S * 2 * LNQ_R * (uint32_t)D * sizeof(T) + 2 * S * 8 + 64;
      { int rc_ = set_max_dynamic_smem((const void*)kern, (int)smem); if (rc_) return rc_; }
      const int blocks = std::min(rows / LNQ_R, num_sms());
      PACI_LAUNCH(kern, blocks, (SETS * LNQ_R + 1) * 32, smem, s, rows, (const T*)x, (const T*)res, g, b, (T*)xsum, (T*)y,
                  mean, rstd);
      return PACI_OK;
    }
  }
  const int nv = ceil_div(D / V, 32);
  const int wpb = 8;
  dim3 grid(ceil_div(rows, wpb)), block(wpb * 32);
#define LN_CASE(N)                                                                                      \
  case N:                                                                                               \
    PACI_LAUNCH((ln_fwd_kernel<T, N>), grid, block, 0, s, rows, D, (const T*)x, (const T*)res, g, b,    \
                (T*)xsum, (T*)y, mean, rstd);                                                           \
    break;
  switch (nv) {
    LN_CASE(1) LN_CASE(2) LN_CASE(3) LN_CASE(4) LN_CASE(5) LN_CASE(6) LN_CASE(7) LN_CASE(8)
    default: return fail(PACI_EINVAL, "layernorm: D=%d too large", D);
  }
#undef LN_CASE
  return PACI_OK;
}

int ln_fwd(int dtype, int rows, int D, const void* x, const void* res, const float* g, const float* b,
           void* xsum, void* y, float* mean, float* rstd, cudaStream_t s) {
  if (rows <= 0) return PACI_OK;
  const double e = dtype == PACI_BF16 ? 2.0 : 4.0;
  ProfScope prof(PC_LN_FWD, 0.0, e * rows * (double)D * (2 + (res != nullptr) + (xsum != nullptr)) + 8.0 * rows, s);
  return dtype == PACI_BF16 ? ln_fwd_t<bf16>(rows, D, x, res, g, b, xsum, y, mean, rstd, s)
                            : ln_fwd_t<float>(rows, D, x, res, g, b, xsum, y, mean, rstd, s);
}

// =========================================================================== LayerNorm backward
// dx = dres + rstd * (g*dy - mean(g*dy) - xhat * mean(g*dy*xhat)) with the CURRENT gain g (Eq. 1) and
// xhat recomputed from the stashed x, mean, rstd (no parameter involved).  Two kernels, both HBM-bound:
//   ln_bwd_dx_kernel    one warp per row, the row in registers, two warp-shuffle reductions; writes dx.
//   ln_bwd_cols_kernel  the three column reductions Gg += sum dy*xhat, Gb += sum dy, Gcol += sum dx:
//                       a thread owns one 16-byte column vector, a block walks its share of the rows four
//                       at a time (independent loads in flight), the block's four row groups meet in shared
//                       memory, then one global atomic per column per block.  It re-reads dy, x and dx, which
//                       the first kernel has just pulled through the 126 MB L2.
// (A single kernel holding the 3 x D/32 column partials per lane needed > 200 registers: one 8-warp CTA per
// SM and 0.13 of HBM peak.)
template <typename T, int NV>
__global__ void __launch_bounds__(256, 3) ln_bwd_dx_kernel(int rows, int D, const T* __restrict__ dy,
                                                           const T* __restrict__ x, const float* __restrict__ mean,
                                                           const float* __restrict__ rstd,
                                                           const float* __restrict__ g, const T* __restrict__ dres,
                                                           T* __restrict__ dx) {
  PACI_PDL_SYNC;
  constexpr int V = Vec<T>::N;
  const int lane = threadIdx.x & 31;
  const int row = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (row >= rows) return;
  const int nvec = D / V;
  const size_t base = (size_t)row * D;
  // the row stays PACKED in registers (3 x NV x 4 registers) and is unpacked once per pass, which leaves
  // room for three 8-warp CTAs per SM: more rows, i.e. more bytes, in flight
  uint4 rdy[NV], rx[NV], rr[NV];
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    const int c = lane + 32 * i;
    if (c < nvec) {
      rdy[i] = load_raw<T>(dy + base + (size_t)c * V);
      rx[i] = load_raw<T>(x + base + (size_t)c * V);
      if (dres != nullptr) rr[i] = load_raw<T>(dres + base + (size_t)c * V);
    }
  }
  const float mu = mean[row], rs = rstd[row];
  float s1 = 0.f, s2 = 0.f;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    const int c = lane + 32 * i;
    if (c < nvec) {
      float gg[V], dyv[V], xv[V];
      load_f32<V>(g + (size_t)c * V, gg);
      unpack_raw<T>(rdy[i], dyv);
      unpack_raw<T>(rx[i], xv);
#pragma unroll
      for (int j = 0; j < V; ++j) {
        const float gd = dyv[j] * gg[j];
        s1 += gd;
        s2 += gd * ((xv[j] - mu) * rs);
      }
    }
  }
  const float invD = 1.f / (float)D;
  s1 = warp_sum(s1) * invD;
  s2 = warp_sum(s2) * invD;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    const int c = lane + 32 * i;
    if (c < nvec) {
      float gg[V], dyv[V], xv[V], o[V];
      load_f32<V>(g + (size_t)c * V, gg);
      unpack_raw<T>(rdy[i], dyv);
      unpack_raw<T>(rx[i], xv);
#pragma unroll
      for (int j = 0; j < V; ++j) o[j] = rs * (dyv[j] * gg[j] - s1 - ((xv[j] - mu) * rs) * s2);
      if (dres != nullptr) {
        float r[V];
        unpack_raw<T>(rr[i], r);
#pragma unroll
        for (int j = 0; j < V; ++j) o[j] += r[j];
      }
      store_vec<T>(dx + base + (size_t)c * V, o);
    }
  }
}

// 1024-thread blocks, one per SM: every column then receives only ~148 global atomics (444 small blocks put 444
// serialized L2 atomics on each 16-byte address, which cost more than streaming the 50 MB)
constexpr int LNC_TX = 128, LNC_TY = 8, LNC_U = 2;
template <typename T>
__global__ void __launch_bounds__(LNC_TX * LNC_TY, 1) ln_bwd_cols_kernel(int rows, int D, const T* __restrict__ dy,
                                                                       const T* __restrict__ x,
                                                                       const float* __restrict__ mean,
                                                                       const float* __restrict__ rstd,
                                                                       const T* __restrict__ dx, float* __restrict__ Gg,
                                                                       float* __restrict__ Gb, float* __restrict__ Gcol) {
  PACI_PDL_SYNC;
  constexpr int V = Vec<T>::N;
  __shared__ __align__(16) float red[3][LNC_TX * V];
  const int tx = threadIdx.x, ty = threadIdx.y;
  const int c = (blockIdx.x * LNC_TX + tx) * V;
  const bool live = c < D;
  for (int i = ty * LNC_TX + tx; i < 3 * LNC_TX * V; i += LNC_TX * LNC_TY) (&red[0][0])[i] = 0.f;
  __syncthreads();
  float ag[V], ab[V], ac[V];
#pragma unroll
  for (int j = 0; j < V; ++j) ag[j] = ab[j] = ac[j] = 0.f;
  const int stride = gridDim.y * LNC_TY;
  if (live) {
    for (int r0 = blockIdx.y * LNC_TY + ty; r0 < rows; r0 += LNC_U * stride) {
      uint4 rdy[LNC_U], rx[LNC_U], rdx[LNC_U];
      float mu[LNC_U], rs[LNC_U];
#pragma unroll
      for (int u = 0; u < LNC_U; ++u) {
        const int r = r0 + u * stride;
        if (r < rows) {
          const size_t off = (size_t)r * D + c;
          rdy[u] = load_raw<T>(dy + off);
          rx[u] = load_raw<T>(x + off);
          if (Gcol != nullptr) rdx[u] = load_raw<T>(dx + off);
          mu[u] = __ldg(mean + r);
          rs[u] = __ldg(rstd + r);
        }
      }
#pragma unroll
      for (int u = 0; u < LNC_U; ++u) {
        if (r0 + u * stride < rows) {
          float dyv[V], xv[V];
          unpack_raw<T>(rdy[u], dyv);
          unpack_raw<T>(rx[u], xv);
#pragma unroll
          for (int j = 0; j < V; ++j) {
            ag[j] += dyv[j] * ((xv[j] - mu[u]) * rs[u]);
            ab[j] += dyv[j];
          }
          if (Gcol != nullptr) {
            float dxv[V];
            unpack_raw<T>(rdx[u], dxv);
#pragma unroll
            for (int j = 0; j < V; ++j) ac[j] += dxv[j];
          }
        }
      }
    }
#pragma unroll
    for (int j = 0; j < V; ++j) {
      atomicAdd(&red[0][tx * V + j], ag[j]);
      atomicAdd(&red[1][tx * V + j], ab[j]);
      if (Gcol != nullptr) atomicAdd(&red[2][tx * V + j], ac[j]);
    }
  }
  __syncthreads();
  // one vector atomic per 4 columns per block (D % 4 == 0, G tensors are 16-byte aligned in the arena)
  for (int i = (ty * LNC_TX + tx) * 4; i < LNC_TX * V; i += LNC_TX * LNC_TY * 4) {
    const int col = blockIdx.x * LNC_TX * V + i;
    if (col < D) {
      red_add_v4(Gg + col, red[0][i], red[0][i + 1], red[0][i + 2], red[0][i + 3]);
      red_add_v4(Gb + col, red[1][i], red[1][i + 1], red[1][i + 2], red[1][i + 3]);
      if (Gcol != nullptr) red_add_v4(Gcol + col, red[2][i], red[2][i + 1], red[2][i + 2], red[2][i + 3]);
    }
  }
}

// Single-pass variant (D = NW x 32 x V, NW <= 8 warps per row): a block of NW warps owns a stream of rows and
// handles LNF_R of them per iteration; a lane owns ONE 16-byte column vector, so the three column partials are
// 3 V registers (not 3 D/32 as in a warp-per-row kernel) and dy, x, dres are read exactly once.  The row sums
// mean(g dy), mean(g dy xhat) cross the NW warps through shared memory (one barrier per LNF_R rows, double-
// buffered).  Per block, one vector atomic per 4 columns at the end.
constexpr int LNF_R = 4;
template <typename T, int NW>
__global__ void __launch_bounds__(NW * 32) ln_bwd_fused_kernel(int rows, int D, const T* __restrict__ dy,
                                                               const T* __restrict__ x, const float* __restrict__ mean,
                                                               const float* __restrict__ rstd,
                                                               const float* __restrict__ g, const T* __restrict__ dres,
                                                               T* __restrict__ dx, float* __restrict__ Gg,
                                                               float* __restrict__ Gb, float* __restrict__ Gcol) {
  PACI_PDL_SYNC;
  constexpr int V = Vec<T>::N;
  __shared__ float part[2][LNF_R][2][NW];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int c = (w * 32 + lane) * V;                      // this lane's columns
  float gg[V], ag[V], ab[V], ac[V];
  load_f32<V>(g + c, gg);
#pragma unroll
  for (int j = 0; j < V; ++j) ag[j] = ab[j] = ac[j] = 0.f;
  const float invD = 1.f / (float)D;
  int buf = 0;
  for (int r0 = blockIdx.x * LNF_R; r0 < rows; r0 += gridDim.x * LNF_R, buf ^= 1) {
    uint4 rdy[LNF_R], rx[LNF_R], rr[LNF_R];
    float mu[LNF_R], rs[LNF_R];
#pragma unroll
    for (int u = 0; u < LNF_R; ++u) {
      const int r = r0 + u;
      if (r < rows) {
        const size_t off = (size_t)r * D + c;
        rdy[u] = load_raw<T>(dy + off);
        rx[u] = load_raw<T>(x + off);
        if (dres != nullptr) rr[u] = load_raw<T>(dres + off);
        mu[u] = __ldg(mean + r);
        rs[u] = __ldg(rstd + r);
      }
    }
#pragma unroll
    for (int u = 0; u < LNF_R; ++u) {
      float s1 = 0.f, s2 = 0.f;
      if (r0 + u < rows) {
        float dyv[V], xv[V];
        unpack_raw<T>(rdy[u], dyv);
        unpack_raw<T>(rx[u], xv);
#pragma unroll
        for (int j = 0; j < V; ++j) {
          const float gd = dyv[j] * gg[j];
          s1 += gd;
          s2 += gd * ((xv[j] - mu[u]) * rs[u]);
        }
      }
      s1 = warp_sum(s1);
      s2 = warp_sum(s2);
      if (lane == 0) { part[buf][u][0][w] = s1; part[buf][u][1][w] = s2; }
    }
    __syncthreads();
#pragma unroll
    for (int u = 0; u < LNF_R; ++u) {
      const int r = r0 + u;
      if (r < rows) {
        float s1 = 0.f, s2 = 0.f;
#pragma unroll
        for (int k = 0; k < NW; ++k) { s1 += part[buf][u][0][k]; s2 += part[buf][u][1][k]; }
        s1 *= invD;
        s2 *= invD;
        float dyv[V], xv[V], o[V];
        unpack_raw<T>(rdy[u], dyv);
        unpack_raw<T>(rx[u], xv);
#pragma unroll
        for (int j = 0; j < V; ++j) {
          const float xh = (xv[j] - mu[u]) * rs[u];
          o[j] = rs[u] * (dyv[j] * gg[j] - s1 - xh * s2);
          ag[j] += dyv[j] * xh;
          ab[j] += dyv[j];
        }
        if (dres != nullptr) {
          float rv[V];
          unpack_raw<T>(rr[u], rv);
#pragma unroll
          for (int j = 0; j < V; ++j) o[j] += rv[j];
        }
        store_vec<T>(dx + (size_t)r * D + c, o);
        if (Gcol != nullptr) {
#pragma unroll
          for (int j = 0; j < V; ++j) ac[j] += to_f(from_f<T>(o[j]));   // sum of what was stored
        }
      }
    }
  }
#pragma unroll
  for (int j = 0; j < V; j += 4) {
    red_add_v4(Gg + c + j, ag[j], ag[j + 1], ag[j + 2], ag[j + 3]);
    red_add_v4(Gb + c + j, ab[j], ab[j + 1], ab[j + 2], ab[j + 3]);
    if (Gcol != nullptr) red_add_v4(Gcol + c + j, ac[j], ac[j + 1], ac[j + 2], ac[j + 3]);
  }
}

// Pipelined variant of the single-pass kernel: one producer thread per block streams LNP_R-row groups of dy, x
// (and dres) plus their mean / rstd into an S-stage shared-memory ring with bulk async copies (one copy per tensor
// per group: the rows of a group are contiguous), so the NW compute warps never wait on a global load -- the
// register-resident version above keeps the loads and the arithmetic of one group in series (26 us, 24% of DRAM
// peak at 20% occupancy).  The compute warps pull a group into registers, hand the stage back at once, and carry
// on exactly as above.  Requires rows % LNP_R == 0 and 16-byte aligned mean / rstd.
constexpr int LNP_R = 4;
__device__ __forceinline__ uint32_t lnp_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void lnp_bulk_load(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(lnp_smem_u32(dst)), "l"(src), "r"(bytes), "r"(lnp_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void lnp_wait(uint64_t* bar, uint32_t parity) {
  tc::mbar_wait_many(bar, parity, 40);                    // parked try_wait; traps after 4 s instead of hanging
}

template <typename T, int NW, int S, int SETS, int RS>
__global__ void __launch_bounds__((SETS * NW + 1) * 32, SETS > 1 ? 1 : 2) ln_bwd_pipe_kernel(int rows, int D, const T* __restrict__ dy,
                                                                   const T* __restrict__ x, const float* __restrict__ mean,
                                                                   const float* __restrict__ rstd,
                                                                   const float* __restrict__ g, const T* __restrict__ dres,
                                                                   T* __restrict__ dx, float* __restrict__ Gg,
                                                                   float* __restrict__ Gb, float* __restrict__ Gcol) {
  PACI_PDL_SYNC;
  constexpr int V = Vec<T>::N;
  constexpr uint32_t RB = NW * 32 * V * sizeof(T);        // bytes of one row
  constexpr uint32_t TB = LNP_R * RB;                     // one tensor's share of a stage
  constexpr uint32_t STAGE = 3 * TB + 32;                 // dy, x, dres, mean[R], rstd[R]
  extern __shared__ __align__(128) uint8_t lnp_smem[];
  uint64_t* full = reinterpret_cast<uint64_t*>(lnp_smem + S * STAGE);
  uint64_t* empty = full + S;
  float (*part)[LNP_R][2][NW] = reinterpret_cast<float (*)[LNP_R][2][NW]>(empty + S);   // [2 * SETS]
  const int lane = threadIdx.x & 31, w = (threadIdx.x >> 5) % NW, set = (threadIdx.x >> 5) / NW;   // set == SETS: producer
  const int groups = rows / LNP_R;
  if (threadIdx.x == 0) {
    for (int i = 0; i < S; ++i) {
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(lnp_smem_u32(&full[i])), "r"(1));
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(lnp_smem_u32(&empty[i])), "r"(NW));
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (set == SETS) {                                      // producer
    if (lane == 0) {
      uint32_t it = 0;
      for (int gi = blockIdx.x; gi < groups; gi += gridDim.x, ++it) {
        const uint32_t st = it % S;
        lnp_wait(&empty[st], ((it / S) & 1u) ^ 1u);
        uint8_t* base = lnp_smem + st * STAGE;
        const size_t off = (size_t)gi * LNP_R * (NW * 32 * V);
        const uint32_t bytes = (dres != nullptr ? 3u : 2u) * TB + 32u;
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(lnp_smem_u32(&full[st])), "r"(bytes) : "memory");
        lnp_bulk_load(base, dy + off, TB, &full[st]);
        lnp_bulk_load(base + TB, x + off, TB, &full[st]);
        if (dres != nullptr) lnp_bulk_load(base + 2 * TB, dres + off, TB, &full[st]);
        lnp_bulk_load(base + 3 * TB, mean + (size_t)gi * LNP_R, 16, &full[st]);
        lnp_bulk_load(base + 3 * TB + 16, rstd + (size_t)gi * LNP_R, 16, &full[st]);
      }
    }
    return;
  }
  const int c = (w * 32 + lane) * V;                      // this lane's columns
  float gg[V], ag[V], ab[V], ac[V];
  load_f32<V>(g + c, gg);
#pragma unroll
  for (int j = 0; j < V; ++j) ag[j] = ab[j] = ac[j] = 0.f;
  const float invD = 1.f / (float)D;
  // SETS groups of NW compute warps take alternate row groups off the ring (so the shuffle / barrier latency of one
  // group hides behind the others') and walk a group RS rows at a time (registers)
  uint32_t it = set, hb = 0;
  for (int gi = blockIdx.x + set * gridDim.x; gi < groups; gi += SETS * gridDim.x, it += SETS) {
    const uint32_t st = it % S;
    lnp_wait(&full[st], (it / S) & 1u);
    const uint8_t* base = lnp_smem + st * STAGE;
#pragma unroll 1
    for (int h0 = 0; h0 < LNP_R; h0 += RS, hb ^= 1u) {
    const uint32_t buf = set * 2 + hb;
    const int r0 = gi * LNP_R + h0;
    uint4 rdy[RS], rx[RS], rr[RS];
    float mu[RS], rs[RS];
#pragma unroll
    for (int u = 0; u < RS; ++u) {
      const uint32_t o = (h0 + u) * RB + (uint32_t)c * sizeof(T);
      rdy[u] = *reinterpret_cast<const uint4*>(base + o);
      rx[u] = *reinterpret_cast<const uint4*>(base + TB + o);
      if (dres != nullptr) rr[u] = *reinterpret_cast<const uint4*>(base + 2 * TB + o);
      mu[u] = *reinterpret_cast<const float*>(base + 3 * TB + 4 * (h0 + u));
      rs[u] = *reinterpret_cast<const float*>(base + 3 * TB + 16 + 4 * (h0 + u));
    }
    if (h0 + RS == LNP_R) {                               // the group is in registers: hand the stage back
      __syncwarp();
      if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(lnp_smem_u32(&empty[st])) : "memory");
    }
#pragma unroll
    for (int u = 0; u < RS; ++u) {
      float dyv[V], xv[V];
      unpack_raw<T>(rdy[u], dyv);
      unpack_raw<T>(rx[u], xv);
      float s1 = 0.f, s2 = 0.f;
#pragma unroll
      for (int j = 0; j < V; ++j) {
        const float gd = dyv[j] * gg[j];
        s1 += gd;
        s2 += gd * ((xv[j] - mu[u]) * rs[u]);
      }
      s1 = warp_sum(s1);
      s2 = warp_sum(s2);
      if (lane == 0) { part[buf][u][0][w] = s1; part[buf][u][1][w] = s2; }
    }
    asm volatile("bar.sync %0, %1;" ::"r"(1 + set), "n"(NW * 32) : "memory");   // this set's compute warps only
#pragma unroll
    for (int u = 0; u < RS; ++u) {
      float s1 = 0.f, s2 = 0.f;
#pragma unroll
      for (int k = 0; k < NW; ++k) { s1 += part[buf][u][0][k]; s2 += part[buf][u][1][k]; }
      s1 *= invD;
      s2 *= invD;
      float dyv[V], xv[V], o[V];
      unpack_raw<T>(rdy[u], dyv);
      unpack_raw<T>(rx[u], xv);
#pragma unroll
      for (int j = 0; j < V; ++j) {
        const float xh = (xv[j] - mu[u]) * rs[u];
        o[j] = rs[u] * (dyv[j] * gg[j] - s1 - xh * s2);
        ag[j] += dyv[j] * xh;
        ab[j] += dyv[j];
      }
      if (dres != nullptr) {
        float rv[V];
        unpack_raw<T>(rr[u], rv);
#pragma unroll
        for (int j = 0; j < V; ++j) o[j] += rv[j];
      }
      store_vec<T>(dx + (size_t)(r0 + u) * D + c, o);
      if (Gcol != nullptr) {
#pragma unroll
        for (int j = 0; j < V; ++j) ac[j] += to_f(from_f<T>(o[j]));   // sum of what was stored
      }
    }
    }
  }
  // same-address atomics serialise in L2 (~27 cycles each), so the sets first add their partials in shared memory
  // (the ring is drained) and each block issues ONE vector atomic per 4 columns
  if (SETS > 1) {
    float* red = reinterpret_cast<float*>(lnp_smem);      // [SETS - 1][3][D]
    asm volatile("bar.sync 15, %0;" ::"n"(SETS * NW * 32) : "memory");   // every set is done with the ring
    if (set > 0) {
      float* dst = red + (size_t)(set - 1) * 3 * D + c;
#pragma unroll
      for (int j = 0; j < V; ++j) { dst[j] = ag[j]; dst[D + j] = ab[j]; dst[2 * D + j] = ac[j]; }
    }
    asm volatile("bar.sync 15, %0;" ::"n"(SETS * NW * 32) : "memory");
    if (set > 0) return;
#pragma unroll
    for (int q = 0; q < SETS - 1; ++q) {
      const float* src = red + (size_t)q * 3 * D + c;
#pragma unroll
      for (int j = 0; j < V; ++j) { ag[j] += src[j]; ab[j] += src[D + j]; ac[j] += src[2 * D + j]; }
    }
  }
#pragma unroll
  for (int j = 0; j < V; j += 4) {
    red_add_v4(Gg + c + j, ag[j], ag[j + 1], ag[j + 2], ag[j + 3]);
    red_add_v4(Gb + c + j, ab[j], ab[j + 1], ab[j + 2], ab[j + 3]);
    if (Gcol != nullptr) red_add_v4(Gcol + c + j, ac[j], ac[j + 1], ac[j + 2], ac[j + 3]);
  }
}

template <typename T>
static int ln_bwd_t(int rows, int D, const void* dy, const void* x, const float* mean, const float* rstd,
                    const float* g, const void* dres, void* dx, float* Gg, float* Gb, float* Gcol,
                    cudaStream_t s) {
  constexpr int V = Vec<T>::N;
  if (D % V != 0) return fail(PACI_EINVAL, "layernorm_bwd: D=%d not a multiple of %d", D, V);
  if (D % (32 * V) == 0 && D / (32 * V) <= 8 && (uintptr_t)Gg % 16 == 0 && (uintptr_t)Gb % 16 == 0 &&
      (Gcol == nullptr || (uintptr_t)Gcol % 16 == 0)) {
    const int nw = D / (32 * V);
    // the shape the stage runs at (bf16, D = 1024): the bulk-copy pipelined kernel, one block per SM (8-stage ring of
    // 4-row groups = 197 KB, 3 sets of 4 compute warps, 2 rows at a time)
    if constexpr (sizeof(T) == 2) {
      if (nw == 4 && rows % LNP_R == 0 && (uintptr_t)mean % 16 == 0 && (uintptr_t)rstd % 16 == 0 &&
          (uintptr_t)dy % 16 == 0 && (uintptr_t)x % 16 == 0 && (uintptr_t)dres % 16 == 0) {
        // S is a multiple of SETS: every ring stage then belongs to ONE set, so each `full` barrier has a single
        // consumer sequence and a waiter can never be two phases behind it (parity waits cannot tell those apart)
        constexpr int S = 9, SETS = 3;
        static_assert(S % SETS == 0, "one owner set per stage");
        auto kern = ln_bwd_pipe_kernel<T, 4, S, SETS, 2>;
        const uint32_t stage = 3 * LNP_R * (uint32_t)D * sizeof(T) + 32;
        const uint32_t smem = S * stage + 2 * S * 8 + 2 * SETS * LNP_R * 2 * 4 * 4 + 64;
        { int rc_ = set_max_dynamic_smem((const void*)kern, (int)smem); if (rc_) return rc_; }
        const int blocks = std::min(rows / LNP_R, num_sms());
        PACI_LAUNCH(kern, blocks, (4 * SETS + 1) * 32, smem, s, rows, D, (const T*)dy, (const T*)x, mean, rstd, g,
                    (const T*)dres, (T*)dx, Gg, Gb, Gcol);
        return PACI_OK;
      }
    }
    const int blocks = std::min(ceil_div(rows, LNF_R), num_sms() * std::max(1, 16 / nw));
#define LNF_CASE(N)                                                                                      \
  case N:                                                                                                \
    PACI_LAUNCH((ln_bwd_fused_kernel<T, N>), blocks, N * 32, 0, s, rows, D, (const T*)dy, (const T*)x,  \
                mean, rstd, g, (const T*)dres, (T*)dx, Gg, Gb, Gcol);                                    \
    return PACI_OK;
    switch (nw) { LNF_CASE(1) LNF_CASE(2) LNF_CASE(3) LNF_CASE(4) LNF_CASE(5) LNF_CASE(6) LNF_CASE(7) LNF_CASE(8) }
#undef LNF_CASE
  }
  const int nv = ceil_div(D / V, 32);
  const int wpb = 8;
  dim3 grid(ceil_div(rows, wpb)), block(wpb * 32);
#define LNB_CASE(N)                                                                                     \
  case N:                                                                                               \
    PACI_LAUNCH((ln_bwd_dx_kernel<T, N>), grid, block, 0, s, rows, D, (const T*)dy, (const T*)x, mean,  \
                rstd, g, (const T*)dres, (T*)dx);                                                       \
    break;
  switch (nv) {
    LNB_CASE(1) LNB_CASE(2) LNB_CASE(3) LNB_CASE(4) LNB_CASE(5) LNB_CASE(6) LNB_CASE(7) LNB_CASE(8)
    default: return fail(PACI_EINVAL, "layernorm_bwd: D=%d too large", D);
  }
#undef LNB_CASE
  const int gx = ceil_div(D / V, LNC_TX);
  int gy = std::max(1, num_sms() / gx);
  gy = std::min(gy, ceil_div(rows, LNC_TY));
  PACI_LAUNCH((ln_bwd_cols_kernel<T>), dim3(gx, gy), dim3(LNC_TX, LNC_TY), 0, s, rows, D, (const T*)dy,
              (const T*)x, mean, rstd, (const T*)dx, Gg, Gb, Gcol);
  return PACI_OK;
}

int ln_bwd(int dtype, int rows, int D, const void* dy, const void* x, const float* mean, const float* rstd,
           const float* g, const void* dres, void* dx, float* Gg, float* Gb, float* Gcol, cudaStream_t s) {
  if (rows <= 0) return PACI_OK;
  const double e = dtype == PACI_BF16 ? 2.0 : 4.0;
  ProfScope prof(PC_LN_BWD, 0.0, e * rows * (double)D * (3 + (dres != nullptr)) + 8.0 * rows, s);
  return dtype == PACI_BF16 ? ln_bwd_t<bf16>(rows, D, dy, x, mean, rstd, g, dres, dx, Gg, Gb, Gcol, s)
                            : ln_bwd_t<float>(rows, D, dy, x, mean, rstd, g, dres, dx, Gg, Gb, Gcol, s);
}

// =========================================================================== GELU
// tanh: accurate tanhf in fp32 mode (1e-5 parity gate); in bf16 mode the single-instruction MUFU.TANH
// (max abs error ~5e-4, below the bf16 rounding of the result) keeps the kernels HBM-bound, not ALU-bound.
template <typename T> __device__ __forceinline__ float tanh_t(float u) { return tanhf(u); }
template <> __device__ __forceinline__ float tanh_t<bf16>(float u) { return tanh_fast(u); }
template <typename T> __device__ __forceinline__ float gelu_f(float p) {
  const float u = p * fmaf(GELU_C * GELU_A, p * p, GELU_C);
  const float h = 0.5f * p;
  return fmaf(h, tanh_t<T>(u), h);
}
// gelu'(p) = 0.5 (1 + th) + (1 - th^2) p (0.5 C + 1.5 C A p^2), th = tanh(p (C + C A p^2)): the same expression as
// 0.5 (1 + th) + 0.5 p (1 - th^2) C (1 + 3 A p^2), arranged as eight FMA-class operations and the tanh
template <typename T> __device__ __forceinline__ float dgelu_f(float p) {
  const float q = p * p;
  const float th = tanh_t<T>(p * fmaf(GELU_C * GELU_A, q, GELU_C));
  const float pw = p * fmaf(1.5f * GELU_C * GELU_A, q, 0.5f * GELU_C);
  return fmaf(fmaf(-th, th, 1.f), pw, fmaf(0.5f, th, 0.5f));
}

// Two elements at a time on sm_100's packed fp32 pairs (FMUL2 / FFMA2: one issue slot for both): the GELU backward
// kernel is partly ALU-bound, and the derivative is most of its arithmetic.  Same expression as dgelu_f<bf16>.
__device__ __forceinline__ unsigned long long f2_pack(float lo, float hi) {
  unsigned long long r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void f2_unpack(unsigned long long v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ unsigned long long f2_mul(unsigned long long a, unsigned long long b) {
  unsigned long long r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ unsigned long long f2_fma(unsigned long long a, unsigned long long b, unsigned long long c) {
  unsigned long long r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}
// (v0, v1) *= gelu'(p0), gelu'(p1)
__device__ __forceinline__ void mul_dgelu2_bf16(float& v0, float& v1, float p0, float p1) {
  const unsigned long long p = f2_pack(p0, p1);
  const unsigned long long q = f2_mul(p, p);
  const unsigned long long u = f2_mul(p, f2_fma(f2_pack(GELU_C * GELU_A, GELU_C * GELU_A), q, f2_pack(GELU_C, GELU_C)));
  float u0, u1;
  f2_unpack(u, u0, u1);
  const unsigned long long th = f2_pack(tanh_fast(u0), tanh_fast(u1));
  const unsigned long long pw = f2_mul(p, f2_fma(f2_pack(1.5f * GELU_C * GELU_A, 1.5f * GELU_C * GELU_A), q,
                                                 f2_pack(0.5f * GELU_C, 0.5f * GELU_C)));
  const unsigned long long one = f2_pack(1.f, 1.f), half = f2_pack(0.5f, 0.5f);
  const unsigned long long nth = f2_mul(th, f2_pack(-1.f, -1.f));
  const unsigned long long d = f2_fma(f2_fma(nth, th, one), pw, f2_fma(half, th, half));
  f2_unpack(f2_mul(f2_pack(v0, v1), d), v0, v1);
}

template <typename T>
__global__ void __launch_bounds__(256) gelu_fwd_kernel(size_t nvec, const T* __restrict__ p, T* __restrict__ out) {
  PACI_PDL_SYNC;
  constexpr int V = Vec<T>::N;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
    float v[V];
    load_vec<T>(p + i * V, v);
#pragma unroll
    for (int j = 0; j < V; ++j) v[j] = gelu_f<T>(v[j]);
    store_vec<T>(out + i * V, v);
  }
}

int gelu_fwd(int dtype, size_t n, const void* p, void* out, cudaStream_t s) {
  if (n == 0) return PACI_OK;
  ProfScope prof(PC_GELU_FWD, 0.0, (dtype == PACI_BF16 ? 2.0 : 4.0) * 2.0 * (double)n, s);
  const int V = dtype == PACI_BF16 ? 8 : 4;
  if (n % V) return fail(PACI_EINVAL, "gelu: n not a multiple of %d", V);
  const size_t nvec = n / V;
  int blocks = (int)std::min<size_t>((nvec + 255) / 256, (size_t)num_sms() * 16);
  if (dtype == PACI_BF16) PACI_LAUNCH(gelu_fwd_kernel<bf16>, blocks, 256, 0, s, nvec, (const bf16*)p, (bf16*)out);
  else PACI_LAUNCH(gelu_fwd_kernel<float>, blocks, 256, 0, s, nvec, (const float*)p, (float*)out);
  return PACI_OK;
}

// Column-slab kernel shared by gelu_bwd and colsum: a thread owns one 16-byte column vector, a block of
// CS_TX x CS_TY threads walks its share of the rows four at a time (independent 16-byte loads in flight),
// partial column sums stay in registers, the block's CS_TY row groups meet in shared memory, and the block
// ends with ONE vector atomic (red.global.add.v4.f32) per 4 columns.  (One scalar atomic per column per
// 128-thread block put ~3000 serialized L2 atomics on every 32-byte sector of G: 0.15 of HBM peak.)
constexpr int CS_TX = 64, CS_TY = 8, CS_U = 4;
template <typename T, bool GELU>
__global__ void __launch_bounds__(CS_TX * CS_TY, 2) colslab_kernel(int rows, int cols, const T* __restrict__ a,
                                                                 const T* __restrict__ p, T* __restrict__ out,
                                                                 float* __restrict__ G) {
  PACI_PDL_SYNC;
  constexpr int V = Vec<T>::N;
  __shared__ __align__(16) float red[CS_TX * V];
  const int tx = threadIdx.x, ty = threadIdx.y;
  const int c = (blockIdx.x * CS_TX + tx) * V;
  const bool live = c < cols;
  if (G != nullptr) {
    for (int i = ty * CS_TX + tx; i < CS_TX * V; i += CS_TX * CS_TY) red[i] = 0.f;
    __syncthreads();
  }
  float acc[V];
#pragma unroll
  for (int j = 0; j < V; ++j) acc[j] = 0.f;
  const int stride = gridDim.y * CS_TY;
  if (live) {
    for (int r0 = blockIdx.y * CS_TY + ty; r0 < rows; r0 += CS_U * stride) {
      uint4 rv[CS_U], rp[CS_U];                        // packed: 8 registers per row instead of 2 V
#pragma unroll
      for (int u = 0; u < CS_U; ++u) {
        const int r = r0 + u * stride;
        if (r < rows) {
          const size_t off = (size_t)r * cols + c;
          rv[u] = load_raw<T>(a + off);
          if (GELU) rp[u] = load_raw<T>(p + off);
        }
      }
#pragma unroll
      for (int u = 0; u < CS_U; ++u) {
        const int r = r0 + u * stride;
        if (r < rows) {
          float v[V];
          unpack_raw<T>(rv[u], v);
          if (GELU) {
            float pv[V];
            unpack_raw<T>(rp[u], pv);
            if constexpr (sizeof(T) == 2) {
#pragma unroll
              for (int j = 0; j < V; j += 2) mul_dgelu2_bf16(v[j], v[j + 1], pv[j], pv[j + 1]);
            } else {
#pragma unroll
              for (int j = 0; j < V; ++j) v[j] *= dgelu_f<T>(pv[j]);
            }
            store_vec<T>(out + (size_t)r * cols + c, v);
#pragma unroll
            for (int j = 0; j < V; ++j) v[j] = to_f(from_f<T>(v[j]));  // sum what was stored
          }
#pragma unroll
          for (int j = 0; j < V; ++j) acc[j] += v[j];
        }
      }
    }
  }
  if (G == nullptr) return;
  if (live) {
#pragma unroll
    for (int j = 0; j < V; ++j) atomicAdd(&red[tx * V + j], acc[j]);
  }
  __syncthreads();
  for (int i = (ty * CS_TX + tx) * 4; i < CS_TX * V; i += CS_TX * CS_TY * 4) {
    const int col = blockIdx.x * CS_TX * V + i;
    if (col < cols) red_add_v4(G + col, red[i], red[i + 1], red[i + 2], red[i + 3]);   // cols % 4 == 0
  }
}

template <bool GELU>
static int colslab(int dtype, int rows, int cols, const void* a, const void* p, void* out, float* G,
                   cudaStream_t s) {
  if (rows <= 0 || cols <= 0) return PACI_OK;
  const int V = dtype == PACI_BF16 ? 8 : 4;
  if (cols % V) return fail(PACI_EINVAL, "colslab: cols=%d not a multiple of %d", cols, V);
  if (G != nullptr && (uintptr_t)G % 16) return fail(PACI_EINVAL, "colslab: G not 16-byte aligned");
  const int gx = ceil_div(cols / V, CS_TX);
  int gy = std::max(1, num_sms() * 4 / gx);
  gy = std::min(gy, ceil_div(rows, CS_TY));
  dim3 grid(gx, gy), block(CS_TX, CS_TY);
  if (dtype == PACI_BF16)
    PACI_LAUNCH((colslab_kernel<bf16, GELU>), grid, block, 0, s, rows, cols, (const bf16*)a, (const bf16*)p,
                (bf16*)out, G);
  else
    PACI_LAUNCH((colslab_kernel<float, GELU>), grid, block, 0, s, rows, cols, (const float*)a,
                (const float*)p, (float*)out, G);
  return PACI_OK;
}

int gelu_bwd(int dtype, int rows, int cols, const void* dg, const void* p, void* dp, float* Gbias,
             cudaStream_t s) {
  ProfScope prof(PC_GELU_BWD, 0.0, (dtype == PACI_BF16 ? 2.0 : 4.0) * 3.0 * rows * (double)cols, s);
  return colslab<true>(dtype, rows, cols, dg, p, dp, Gbias, s);
}
int colsum(int dtype, int rows, int cols, const void* x, float* G, cudaStream_t s) {
  ProfScope prof(PC_COLSUM, 0.0, (dtype == PACI_BF16 ? 2.0 : 4.0) * rows * (double)cols, s);
  return colslab<false>(dtype, rows, cols, x, nullptr, nullptr, G, s);
}

// =========================================================================== embedding
// A token / target id outside [0, vocab) is clamped (no out-of-bounds access) and raises the stage's sticky
// device error word, which paci_stage_check / paci_pipeline_run report as PACI_EINVAL.
__device__ __forceinline__ int checked_id(int id, int vocab, int64_t* err) {
  if ((unsigned)id < (unsigned)vocab) return id;
  if (err != nullptr) *err = 1;
  return id < 0 ? 0 : vocab - 1;
}
template <typename T>
__global__ void __launch_bounds__(256) embed_fwd_kernel(int M, int T_, int D, const int32_t* __restrict__ tok,
                                                        const float* __restrict__ wte,
                                                        const float* __restrict__ wpe, T* __restrict__ x,
                                                        int vocab, int64_t* __restrict__ err) {
  PACI_PDL_SYNC;
  constexpr int V = Vec<T>::N;
  const int nvec = D / V;
  const size_t total = (size_t)M * nvec;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    const int row = (int)(i / nvec), c = (int)(i % nvec) * V;
    const int id = checked_id(tok[row], vocab, err), pos = row % T_;
    float a[V], b[V];
    load_f32<V>(wte + (size_t)id * D + c, a);
    load_f32<V>(wpe + (size_t)pos * D + c, b);
#pragma unroll
    for (int j = 0; j < V; ++j) a[j] += b[j];
    store_vec<T>(x + (size_t)row * D + c, a);
  }
}

int embed_fwd(int dtype, int mu, int T_, int D, const int32_t* tok, const float* wte, const float* wpe, void* x,
              int vocab, int64_t* err, cudaStream_t s) {
  ProfScope prof(PC_EMBED, 0.0, ((dtype == PACI_BF16 ? 2.0 : 4.0) + 4.0) * mu * (double)T_ * D + 4.0 * T_ * D, s);
  const int M = mu * T_;
  const int V = dtype == PACI_BF16 ? 8 : 4;
  if (D % V) return fail(PACI_EINVAL, "embed: D=%d", D);
  const size_t total = (size_t)M * (D / V);
  int blocks = (int)std::min<size_t>((total + 255) / 256, (size_t)num_sms() * 16);
  if (dtype == PACI_BF16)
    PACI_LAUNCH(embed_fwd_kernel<bf16>, blocks, 256, 0, s, M, T_, D, tok, wte, wpe, (bf16*)x, vocab, err);
  else
    PACI_LAUNCH(embed_fwd_kernel<float>, blocks, 256, 0, s, M, T_, D, tok, wte, wpe, (float*)x, vocab, err);
  return PACI_OK;
}

// Gwte[tok] += dx (fp32 vector atomics: red.global.add.v4.f32), Gwpe[t] += sum_b dx[b,t].
template <typename T>
__global__ void __launch_bounds__(256) embed_bwd_wte_kernel(int M, int D, const int32_t* __restrict__ tok,
                                                            const T* __restrict__ dx, float* __restrict__ Gwte,
                                                            int vocab) {
  PACI_PDL_SYNC;
  constexpr int V = Vec<T>::N;
  const int nvec = D / V;
  const size_t total = (size_t)M * nvec;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    const int row = (int)(i / nvec), c = (int)(i % nvec) * V;
    float v[V];
    load_vec<T>(dx + (size_t)row * D + c, v);
    float* dst = Gwte + (size_t)checked_id(tok[row], vocab, nullptr) * D + c;
#pragma unroll
    for (int j = 0; j < V; j += 4)
      asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst + j), "f"(v[j]), "f"(v[j + 1]),
                   "f"(v[j + 2]), "f"(v[j + 3])
                   : "memory");
  }
}
template <typename T>
__global__ void __launch_bounds__(256) embed_bwd_wpe_kernel(int mu, int T_, int D, const T* __restrict__ dx,
                                                            float* __restrict__ Gwpe) {
  PACI_PDL_SYNC;
  constexpr int V = Vec<T>::N;
  const int nvec = D / V;
  const size_t total = (size_t)T_ * nvec;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    const int t = (int)(i / nvec), c = (int)(i % nvec) * V;
    float acc[V];
#pragma unroll
    for (int j = 0; j < V; ++j) acc[j] = 0.f;
    for (int b = 0; b < mu; ++b) {
      float v[V];
      load_vec<T>(dx + ((size_t)b * T_ + t) * D + c, v);
#pragma unroll
      for (int j = 0; j < V; ++j) acc[j] += v[j];
    }
    float* dst = Gwpe + (size_t)t * D + c;
#pragma unroll
    for (int j = 0; j < V; ++j) dst[j] += acc[j];
  }
}

int embed_bwd(int dtype, int mu, int T_, int D, const int32_t* tok, const void* dx, float* Gwte, float* Gwpe,
              int vocab, cudaStream_t s) {
  // dx read twice (wte scatter, wpe reduction) + fp32 read-modify-write of the touched rows
  ProfScope prof(PC_EMBED, 0.0, ((dtype == PACI_BF16 ? 2.0 : 4.0) * 2.0 + 8.0) * mu * (double)T_ * D + 8.0 * T_ * D, s);
  const int M = mu * T_;
  const int V = dtype == PACI_BF16 ? 8 : 4;
  if (D % V) return fail(PACI_EINVAL, "embed_bwd: D=%d", D);
  const size_t t1 = (size_t)M * (D / V), t2 = (size_t)T_ * (D / V);
  int b1 = (int)std::min<size_t>((t1 + 255) / 256, (size_t)num_sms() * 16);
  int b2 = (int)std::min<size_t>((t2 + 255) / 256, (size_t)num_sms() * 16);
  if (dtype == PACI_BF16) {
    PACI_LAUNCH(embed_bwd_wte_kernel<bf16>, b1, 256, 0, s, M, D, tok, (const bf16*)dx, Gwte, vocab);
    PACI_LAUNCH(embed_bwd_wpe_kernel<bf16>, b2, 256, 0, s, mu, T_, D, (const bf16*)dx, Gwpe);
  } else {
    PACI_LAUNCH(embed_bwd_wte_kernel<float>, b1, 256, 0, s, M, D, tok, (const float*)dx, Gwte, vocab);
    PACI_LAUNCH(embed_bwd_wpe_kernel<float>, b2, 256, 0, s, mu, T_, D, (const float*)dx, Gwpe);
  }
  return PACI_OK;
}

// =========================================================================== softmax cross-entropy
// One block per token row: pass 1 reads the row (online max / sum of exp), pass 2 re-reads it (L2
// hit: a row is <= 100 KB) and overwrites it with dz = (softmax - onehot) / rows.  Padding columns
// [V, ldz) are written as 0 so that the following GEMMs can contract over ldz.
template <typename T> __device__ __forceinline__ float exp_t(float x);
template <> __device__ __forceinline__ float exp_t<float>(float x) { return expf(x); }     // 1e-5 parity mode
template <> __device__ __forceinline__ float exp_t<bf16>(float x) { return __expf(x); }

__device__ __forceinline__ float ex2_fast(float x) {
  float r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

// bf16 mode.  The generic kernel below spends ~18 instructions per logit (a bounds test, a subtract, a multiply and a
// select around each of its two exponentials): it was issue-bound at 0.44 of the HBM peak.  Here every constant is
// folded into the exponent -- pass 1 adds exp2(z log2e - max log2e), pass 2 writes exp2(z log2e + K) with
// K = -max log2e + log2(1 / (sum rows)), i.e. softmax / rows in ONE FFMA + MUFU per logit -- the column bound is
// tested per 16-byte vector (only the row's last vectors straddle V), and the one-hot is subtracted from the single
// vector that holds the target.  Same two passes over the row (the second read hits L2), same outputs.
__global__ void __launch_bounds__(512) softmax_ce_bf16_kernel(int rows, int V_, int ldz, bf16* __restrict__ z,
                                                              const int32_t* __restrict__ tgt,
                                                              float* __restrict__ loss, int64_t* __restrict__ err) {
  PACI_PDL_SYNC;
  constexpr int V = 8;
  constexpr float L2E = 1.4426950408889634f;
  __shared__ float red_m[16], red_s[16];
  __shared__ float sh_max, sh_sum;
  const int row = blockIdx.x;
  bf16* zr = z + (size_t)row * ldz;
  const int nvec = ldz / V, nfull = V_ / V;              // vectors [0, nfull) lie entirely inside [0, V_)
  float mx = -INFINITY, sum = 0.f;
  for (int i = threadIdx.x; i < nvec; i += blockDim.x) {
    float v[V];
    load_vec<bf16>(zr + (size_t)i * V, v);
    if (i >= nfull) {
#pragma unroll
      for (int j = 0; j < V; ++j)
        if (i * V + j >= V_) v[j] = -INFINITY;
    }
    const float lm = fmaxf(fmaxf(fmaxf(v[0], v[1]), fmaxf(v[2], v[3])), fmaxf(fmaxf(v[4], v[5]), fmaxf(v[6], v[7])));
    if (lm > mx) {
      sum *= ex2_fast((mx - lm) * L2E);                  // mx = -inf on the first vector: exp2(-inf) = 0
      mx = lm;
    }
    if (mx != -INFINITY) {                               // (a vector of padding only: nothing to add)
      const float nm = -mx * L2E;
      float s0 = 0.f, s1 = 0.f;
#pragma unroll
      for (int j = 0; j < V; j += 2) {
        s0 += ex2_fast(fmaf(v[j], L2E, nm));
        s1 += ex2_fast(fmaf(v[j + 1], L2E, nm));
      }
      sum += s0 + s1;
    }
  }
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const float wm = warp_max(mx);
  const float ws = warp_sum(mx == -INFINITY ? 0.f : sum * ex2_fast((mx - wm) * L2E));
  if (lane == 0) { red_m[w] = wm; red_s[w] = ws; }
  __syncthreads();
  if (w == 0) {
    const int nw = blockDim.x >> 5;
    const float m2 = lane < nw ? red_m[lane] : -INFINITY;
    const float s2 = lane < nw ? red_s[lane] : 0.f;
    const float bm = warp_max(m2);
    const float bs = warp_sum(m2 == -INFINITY ? 0.f : s2 * ex2_fast((m2 - bm) * L2E));
    if (lane == 0) { sh_max = bm; sh_sum = bs; }
  }
  __syncthreads();
  const float bm = sh_max, scale = 1.f / (float)rows;
  const float K = fmaf(-bm, L2E, log2f(scale / sh_sum));
  const int t = checked_id(tgt[row], V_, threadIdx.x == 0 ? err : nullptr);
  if (threadIdx.x == 0) {
    const float zt = to_f(zr[t]);
    atomicAdd(loss, (logf(sh_sum) + bm - zt) * scale);
  }
  __syncthreads();  // zr[t] read before anyone overwrites it
  const int tv = t / V, tj = t % V;
  for (int i = threadIdx.x; i < nvec; i += blockDim.x) {
    float v[V];
    load_vec<bf16>(zr + (size_t)i * V, v);
#pragma unroll
    for (int j = 0; j < V; ++j) v[j] = ex2_fast(fmaf(v[j], L2E, K));
    if (i >= nfull) {
#pragma unroll
      for (int j = 0; j < V; ++j)
        if (i * V + j >= V_) v[j] = 0.f;
    }
    if (i == tv) {
#pragma unroll
      for (int j = 0; j < V; ++j)
        if (j == tj) v[j] -= scale;
    }
    store_vec<bf16>(zr + (size_t)i * V, v);
  }
}

template <typename T>
__global__ void __launch_bounds__(512) softmax_ce_kernel(int rows, int V_, int ldz, T* __restrict__ z,
                                                         const int32_t* __restrict__ tgt,
                                                         float* __restrict__ loss, int64_t* __restrict__ err) {
  PACI_PDL_SYNC;
  constexpr int V = Vec<T>::N;
  __shared__ float red_m[16], red_s[16];
  __shared__ float sh_max, sh_sum;
  const int row = blockIdx.x;
  T* zr = z + (size_t)row * ldz;
  const int nvec = ldz / V;
  float mx = -INFINITY, sum = 0.f;
  for (int i = threadIdx.x; i < nvec; i += blockDim.x) {
    float v[V];
    load_vec<T>(zr + (size_t)i * V, v);
    float lm = -INFINITY;
#pragma unroll
    for (int j = 0; j < V; ++j)
      if (i * V + j < V_) lm = fmaxf(lm, v[j]);
    if (lm > mx) {
      sum *= exp_t<T>(mx - lm);
      mx = lm;
    }
#pragma unroll
    for (int j = 0; j < V; ++j)
      if (i * V + j < V_) sum += exp_t<T>(v[j] - mx);
  }
  // block reduce (max, sum) pairs
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  float wm = warp_max(mx);
  float ws = warp_sum(mx == -INFINITY ? 0.f : sum * exp_t<T>(mx - wm));
  if (lane == 0) { red_m[w] = wm; red_s[w] = ws; }
  __syncthreads();
  if (w == 0) {
    const int nw = blockDim.x >> 5;
    float m2 = lane < nw ? red_m[lane] : -INFINITY;
    float s2 = lane < nw ? red_s[lane] : 0.f;
    const float bm = warp_max(m2);
    const float bs = warp_sum(m2 == -INFINITY ? 0.f : s2 * exp_t<T>(m2 - bm));
    if (lane == 0) { sh_max = bm; sh_sum = bs; }
  }
  __syncthreads();
  const float bm = sh_max, inv = 1.f / sh_sum, scale = 1.f / (float)rows;
  const int t = checked_id(tgt[row], V_, threadIdx.x == 0 ? err : nullptr);
  if (threadIdx.x == 0) {
    const float zt = to_f(zr[t]);
    atomicAdd(loss, (logf(sh_sum) + bm - zt) * scale);
  }
  __syncthreads();  // zr[t] read before anyone overwrites it
  for (int i = threadIdx.x; i < nvec; i += blockDim.x) {
    float v[V];
    load_vec<T>(zr + (size_t)i * V, v);
#pragma unroll
    for (int j = 0; j < V; ++j) {
      const int c = i * V + j;
      float p = c < V_ ? exp_t<T>(v[j] - bm) * inv : 0.f;
      if (c == t) p -= 1.f;
      v[j] = p * scale;
    }
    store_vec<T>(zr + (size_t)i * V, v);
  }
}

int softmax_ce(int dtype, int rows, int V_, int ldz, void* z, const int32_t* tgt, float* loss, int64_t* err,
               cudaStream_t s) {
  ProfScope prof(PC_SOFTMAX_CE, 0.0, (dtype == PACI_BF16 ? 2.0 : 4.0) * 2.0 * rows * (double)ldz, s);
  const int V = dtype == PACI_BF16 ? 8 : 4;
  if (ldz % V || ldz < V_) return fail(PACI_EINVAL, "softmax_ce: ldz=%d V=%d", ldz, V_);
  if (dtype == PACI_BF16) PACI_LAUNCH(softmax_ce_bf16_kernel, rows, 512, 0, s, rows, V_, ldz, (bf16*)z, tgt, loss, err);
  else PACI_LAUNCH(softmax_ce_kernel<float>, rows, 512, 0, s, rows, V_, ldz, (float*)z, tgt, loss, err);
  return PACI_OK;
}

// =========================================================================== fused multi-tensor AdamW
// The stage's parameters live in ONE flat fp32 arena laid out [decayed tensors | non-decayed tensors],
// so a single launch covers every tensor (row a20): 34 B/param in bf16 mode (read w,m,v,G; write
// w,m,v,G=0 and the bf16 shadow).  Thread 0 bumps the device version word (Alg. 1 line 17).
__global__ void __launch_bounds__(256) adamw_kernel(size_t n4, size_t n4_decay, float4* __restrict__ w,
                                                    float4* __restrict__ m, float4* __restrict__ v,
                                                    float4* __restrict__ G, uint2* __restrict__ shadow,
                                                    float inv_k, float lr, float beta1, float beta2, float eps,
                                                    float decay_mul, float inv_bc1, float inv_bc2,
                                                    int64_t* version_word) {
  PACI_PDL_SYNC;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
    float4 W = w[i], Mv = m[i], Vv = v[i], Gv = G[i];
    const float dm = i < n4_decay ? decay_mul : 1.f;
    float* wp = reinterpret_cast<float*>(&W);
    float* mp = reinterpret_cast<float*>(&Mv);
    float* vp = reinterpret_cast<float*>(&Vv);
    const float* gp = reinterpret_cast<const float*>(&Gv);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const float g = gp[j] * inv_k;
      float th = wp[j] * dm;
      mp[j] = beta1 * mp[j] + (1.f - beta1) * g;
      vp[j] = beta2 * vp[j] + (1.f - beta2) * g * g;
      th -= lr * (mp[j] * inv_bc1) / (sqrtf(vp[j] * inv_bc2) + eps);
      wp[j] = th;
    }
    w[i] = W; m[i] = Mv; v[i] = Vv;
    G[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (shadow != nullptr) {
      __nv_bfloat162 lo = __floats2bfloat162_rn(W.x, W.y), hi = __floats2bfloat162_rn(W.z, W.w);
      uint2 o;
      o.x = *reinterpret_cast<uint32_t*>(&lo);
      o.y = *reinterpret_cast<uint32_t*>(&hi);
      shadow[i] = o;
    }
  }
  if (version_word != nullptr && blockIdx.x == 0 && threadIdx.x == 0) *version_word += 1;
}

int adamw(size_t n, size_t n_decay, float* w, float* m, float* v, float* G, void* shadow, int k, int64_t t,
          float lr, float beta1, float beta2, float eps, float wd, int64_t* version_word, cudaStream_t s) {
  ProfScope prof(PC_ADAMW, 0.0, (shadow != nullptr ? 34.0 : 32.0) * (double)n, s);
  if (n % 4 || n_decay % 4) return fail(PACI_EINVAL, "adamw: n=%zu n_decay=%zu must be multiples of 4", n, n_decay);
  const double bc1 = 1.0 - std::pow((double)beta1, (double)t), bc2 = 1.0 - std::pow((double)beta2, (double)t);
  const size_t n4 = n / 4;
  int blocks = (int)std::min<size_t>(std::max<size_t>((n4 + 255) / 256, 1), (size_t)num_sms() * 8);
  PACI_LAUNCH(adamw_kernel, blocks, 256, 0, s, n4, n_decay / 4, (float4*)w, (float4*)m, (float4*)v, (float4*)G,
              (uint2*)shadow, 1.f / (float)k, lr, beta1, beta2, eps, 1.f - lr * wd, (float)(1.0 / bc1),
              (float)(1.0 / bc2), version_word);
  return PACI_OK;
}

__global__ void cast_shadow_kernel(size_t n, const float* __restrict__ w, bf16* __restrict__ sh) {
  PACI_PDL_SYNC;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    sh[i] = __float2bfloat16_rn(w[i]);
}
int cast_shadow(size_t n, const float* w, void* shadow, cudaStream_t s) {
  if (n == 0) return PACI_OK;
  ProfScope prof(PC_OTHER, 0.0, 6.0 * (double)n, s);
  int blocks = (int)std::min<size_t>((n + 255) / 256, (size_t)num_sms() * 8);
  PACI_LAUNCH(cast_shadow_kernel, blocks, 256, 0, s, n, w, (bf16*)shadow);
  return PACI_OK;
}

// =========================================================================== dropout
// Philox4x32-10 (Salmon et al., "Parallel random numbers: as easy as 1, 2, 3"): 10 rounds of
//   (c0, c1, c2, c3) <- (hi(M1 c2) ^ c1 ^ k0, lo(M1 c2), hi(M0 c0) ^ c3 ^ k1, lo(M0 c0)),  k += (W0, W1) between rounds.
// The oracle evaluates the same generator on the same counters (oracle/dropout.py), so the masks agree bit for bit.
struct Philox4 { uint32_t v[4]; };
__device__ __forceinline__ Philox4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                                 uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    c0 = hi1 ^ c1 ^ k0; c1 = lo1; c2 = hi0 ^ c3 ^ k1; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  return Philox4{{c0, c1, c2, c3}};
}

template <typename T>
__global__ void __launch_bounds__(256) dropout_kernel(size_t nvec, const T* __restrict__ x, T* __restrict__ out,
                                                      uint32_t thresh, float scale, uint32_t k0, uint32_t k1,
                                                      uint32_t mb, uint32_t site) {
  PACI_PDL_SYNC;
  constexpr int V = Vec<T>::N;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
    float v[V];
    load_vec<T>(x + i * V, v);
#pragma unroll
    for (int q = 0; q < V / 4; ++q) {
      const uint64_t blk = i * (V / 4) + q;                  // element index / 4
      const Philox4 r = philox4x32_10((uint32_t)blk, (uint32_t)(blk >> 32), mb, site, k0, k1);
#pragma unroll
      for (int j = 0; j < 4; ++j) v[4 * q + j] = r.v[j] >= thresh ? v[4 * q + j] * scale : 0.f;
    }
    store_vec<T>(out + i * V, v);
  }
}

int dropout(int dtype, size_t n, const void* x, void* out, float p, uint64_t seed, int64_t mb_id, int site,
            cudaStream_t s) {
  if (n == 0) return PACI_OK;
  if (!(p >= 0.f && p < 1.f)) return fail(PACI_EINVAL, "dropout: p=%f", (double)p);
  ProfScope prof(PC_OTHER, 0.0, (dtype == PACI_BF16 ? 2.0 : 4.0) * 2.0 * (double)n, s);
  const int V = dtype == PACI_BF16 ? 8 : 4;
  if (n % V) return fail(PACI_EINVAL, "dropout: n not a multiple of %d", V);
  const size_t nvec = n / V;
  const uint32_t thresh = (uint32_t)std::min<double>(std::floor((double)p * 4294967296.0), 4294967295.0);
  const float scale = 1.f / (1.f - p);
  int blocks = (int)std::min<size_t>((nvec + 255) / 256, (size_t)num_sms() * 16);
  if (dtype == PACI_BF16)
    PACI_LAUNCH(dropout_kernel<bf16>, blocks, 256, 0, s, nvec, (const bf16*)x, (bf16*)out, thresh, scale,
                (uint32_t)seed, (uint32_t)(seed >> 32), (uint32_t)mb_id, (uint32_t)site);
  else
    PACI_LAUNCH(dropout_kernel<float>, blocks, 256, 0, s, nvec, (const float*)x, (float*)out, thresh, scale,
                (uint32_t)seed, (uint32_t)(seed >> 32), (uint32_t)mb_id, (uint32_t)site);
  return PACI_OK;
}

template <typename T>
__global__ void __launch_bounds__(256) add_vec_kernel(size_t nvec, const T* __restrict__ a, const T* __restrict__ b,
                                                      T* __restrict__ out) {
  PACI_PDL_SYNC;
  constexpr int V = Vec<T>::N;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
    float x[V];
    load_vec<T>(a + i * V, x);
    if (b != nullptr) {
      float y[V];
      load_vec<T>(b + i * V, y);
#pragma unroll
      for (int j = 0; j < V; ++j) x[j] += y[j];
    }
    store_vec<T>(out + i * V, x);
  }
}
int add_vec(int dtype, size_t n, const void* a, const void* b, void* out, cudaStream_t s) {
  if (n == 0) return PACI_OK;
  ProfScope prof(PC_OTHER, 0.0, (dtype == PACI_BF16 ? 2.0 : 4.0) * (double)n * (2 + (b != nullptr)), s);
  const int V = dtype == PACI_BF16 ? 8 : 4;
  if (n % V) return fail(PACI_EINVAL, "add: n not a multiple of %d", V);
  const size_t nvec = n / V;
  int blocks = (int)std::min<size_t>((nvec + 255) / 256, (size_t)num_sms() * 16);
  if (dtype == PACI_BF16)
    PACI_LAUNCH(add_vec_kernel<bf16>, blocks, 256, 0, s, nvec, (const bf16*)a, (const bf16*)b, (bf16*)out);
  else
    PACI_LAUNCH(add_vec_kernel<float>, blocks, 256, 0, s, nvec, (const float*)a, (const float*)b, (float*)out);
  return PACI_OK;
}

__global__ void stamp_kernel(const int64_t* version_word, int64_t* dst) {
  PACI_PDL_SYNC; *dst = *version_word; }
int stamp_version(const int64_t* version_word, int64_t* dst, cudaStream_t s) {
  PACI_LAUNCH(stamp_kernel, 1, 1, 0, s, version_word, dst);
  return PACI_OK;
}

__global__ void split_tokens_kernel(int mu, int T_, const int32_t* __restrict__ src, int32_t* __restrict__ inp,
                                    int32_t* __restrict__ tgt) {
  PACI_PDL_SYNC;
  const int n = mu * T_;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const int b = i / T_, t = i % T_;
    inp[i] = src[(size_t)b * (T_ + 1) + t];
    tgt[i] = src[(size_t)b * (T_ + 1) + t + 1];
  }
}
int split_tokens(int mu, int T_, const int32_t* tok_tp1, int32_t* inp, int32_t* tgt, cudaStream_t s) {
  PACI_LAUNCH(split_tokens_kernel, ceil_div(mu * T_, 256), 256, 0, s, mu, T_, tok_tp1, inp, tgt);
  return PACI_OK;
}

}  // namespace paci
