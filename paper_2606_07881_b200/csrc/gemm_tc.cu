// gemm_tc.cu -- bf16 GEMM on the 5th-generation tensor cores (tcgen05.mma), hand-written for sm_100a.
// Rows a3, a5, a7, a9, a10 (forward, "NT"), a12/a13 (dgrad with the CURRENT weights, "NN") and a14
// (wgrad whose epilogue ADDS into the fp32 accumulator G, "TN", split-K over tokens) of SURVEY.md 8(a).
//
// Structure (one CTA per SM, persistent over work items, 192 threads):
//   warp 0      TMA producer: cp.async.bulk.tensor 2D tiles -> 128B-swizzled shared memory, 4-stage ring
//   warp 1      MMA issuer: one thread issues tcgen05.mma (M=128, N=BLOCK_N, K=16) from shared-memory
//               matrix descriptors; accumulators live in TMEM (2 buffers x BLOCK_N fp32 columns), so the
//               epilogue of tile i overlaps the main loop of tile i+1
//   warps 2-5   epilogue: tcgen05.ld (32 lanes x 32 columns per warp) -> registers -> (+bias, ->bf16)
//               st.global, or red.global.add.v4.f32 into the fp32 accumulator (beta = 1)
// Pipelines: full/empty mbarriers between TMA and MMA (tcgen05.commit frees a stage), tmem_full /
// tmem_empty between MMA and epilogue.
//
// Operand layouts.  "K-major" = contraction index contiguous in memory, "MN-major" = the other index
// contiguous.  Both are staged by TMA with the 128-byte swizzle and described to the tensor core by a
// shared-memory descriptor (start address, LBO, SBO, SWIZZLE_128B) plus the a_major/b_major bits of
// the instruction descriptor, so no operand is ever transposed in memory:
//   NT: A K-major,  B K-major        NN: A K-major,  B MN-major        TN: A MN-major, B MN-major
// K-major tile  [rows][64 k]: one TMA box {64, rows};  SBO = 1024 B (8 rows x 128 B).
// MN-major tile [64 k][64 mn] per box {64, 64}, rows/64 boxes 8 KB apart: LBO = 8192 B, SBO = 1024 B.
#include <cuda.h>

#include <algorithm>
#include <mutex>
#include <unordered_map>

#include "common.cuh"

namespace paci {

namespace {

constexpr int BLOCK_M = 128;
constexpr int BLOCK_K = 64;
constexpr int UMMA_K = 16;
constexpr int STAGES = 4;
constexpr int NUM_THREADS = 192;

// ------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  const uint32_t addr = smem_u32(bar);
  uint32_t done = 0;
  uint32_t spins = 0;
  while (true) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.b32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(addr), "r"(parity)
        : "memory");
    if (done) break;
    if (++spins > (1u << 26)) __trap();   // a protocol bug must fault, not hang the GPU
  }
}
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
      : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                          uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* bar) {   // arrives on bar when all prior MMAs are done
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
        "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
        "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
        "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// Shared-memory matrix descriptor (sm_100 format: start[0,14) | LBO[16,30) | SBO[32,46) | version=1 at 46 |
// layout type [61,64) with SWIZZLE_128B = 2); addresses and offsets in 16-byte units.
__device__ __forceinline__ uint64_t smem_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  uint64_t d = (uint64_t)((saddr & 0x3FFFFu) >> 4);
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFFu) << 16;
  d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFFu) << 32;
  d |= (uint64_t)1 << 46;
  d |= (uint64_t)2 << 61;
  return d;
}

struct Params {
  int M, N, K, ldc;
  int tiles_m, tiles_n, splits, kb_total;
  const float* bias;
  void* C;
};

// ------------------------------------------------------------------ the kernel
template <int BLOCK_N, bool A_MN, bool B_MN, bool ACCUM>
__global__ void __launch_bounds__(NUM_THREADS, 1)
gemm_tc_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const Params p) {
  constexpr uint32_t A_BYTES = BLOCK_M * BLOCK_K * 2, B_BYTES = BLOCK_N * BLOCK_K * 2;
  constexpr uint32_t STAGE_BYTES = A_BYTES + B_BYTES;
  constexpr uint32_t BOX_MN_BYTES = 64 * BLOCK_K * 2;   // one {64 mn, 64 k} box of an MN-major operand
  constexpr uint32_t TMEM_COLS = 2 * BLOCK_N;
  // instruction descriptor: D fp32 (bit 4), A/B bf16 (bits 7, 10), majors (15, 16), N>>3 at 17, M>>4 at 24
  constexpr uint32_t IDESC = (1u << 4) | (1u << 7) | (1u << 10) | ((A_MN ? 1u : 0u) << 15) |
                             ((B_MN ? 1u : 0u) << 16) | ((uint32_t)(BLOCK_N >> 3) << 17) |
                             ((uint32_t)(BLOCK_M >> 4) << 24);

  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  uint64_t* full = (uint64_t*)(smem + STAGES * STAGE_BYTES);
  uint64_t* empty = full + STAGES;
  uint64_t* tfull = empty + STAGES;
  uint64_t* tempty = tfull + 2;
  uint32_t* tmem_slot = (uint32_t*)(tempty + 2);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (int i = 0; i < STAGES; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&tfull[i], 1); mbar_init(&tempty[i], 4); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)),
                 "r"(TMEM_COLS)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  const int n_items = p.tiles_m * p.tiles_n * p.splits;
  const int kb_per = (p.kb_total + p.splits - 1) / p.splits;

  if (warp == 0) {
    if (lane == 0) {
      asm volatile("prefetch.tensormap [%0];" ::"l"(&tmA) : "memory");
      asm volatile("prefetch.tensormap [%0];" ::"l"(&tmB) : "memory");
      uint32_t stage = 0, phase = 0;
      for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        const int tile = item / p.splits, split = item % p.splits;
        const int m0 = (tile % p.tiles_m) * BLOCK_M, n0 = (tile / p.tiles_m) * BLOCK_N;
        const int kb0 = split * kb_per, kb1 = min(kb0 + kb_per, p.kb_total);
        for (int kb = kb0; kb < kb1; ++kb) {
          mbar_wait(&empty[stage], phase ^ 1);
          uint8_t* sa = smem + stage * STAGE_BYTES;
          uint8_t* sb = sa + A_BYTES;
          mbar_expect_tx(&full[stage], STAGE_BYTES);
          const int k0 = kb * BLOCK_K;
          if (A_MN) {
#pragma unroll
            for (int i = 0; i < BLOCK_M / 64; ++i) tma_load_2d(sa + i * BOX_MN_BYTES, &tmA, &full[stage], m0 + i * 64, k0);
          } else {
            tma_load_2d(sa, &tmA, &full[stage], k0, m0);
          }
          if (B_MN) {
#pragma unroll
            for (int i = 0; i < BLOCK_N / 64; ++i) tma_load_2d(sb + i * BOX_MN_BYTES, &tmB, &full[stage], n0 + i * 64, k0);
          } else {
            tma_load_2d(sb, &tmB, &full[stage], k0, n0);
          }
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {
      uint32_t stage = 0, phase = 0, acc = 0, acc_phase = 0;
      for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        const int split = item % p.splits;
        const int kb0 = split * kb_per, kb1 = min(kb0 + kb_per, p.kb_total);
        mbar_wait(&tempty[acc], acc_phase ^ 1);      // epilogue has drained this accumulator
        tc_fence_after();
        const uint32_t tmem_d = tmem_base + acc * BLOCK_N;
        for (int kb = kb0; kb < kb1; ++kb) {
          mbar_wait(&full[stage], phase);
          tc_fence_after();
          const uint32_t sa = smem_u32(smem + stage * STAGE_BYTES), sb = sa + A_BYTES;
#pragma unroll
          for (int j = 0; j < BLOCK_K / UMMA_K; ++j) {
            const uint64_t ad = A_MN ? smem_desc(sa + j * (UMMA_K * 128), BOX_MN_BYTES, 1024)
                                     : smem_desc(sa + j * (UMMA_K * 2), 16, 1024);
            const uint64_t bd = B_MN ? smem_desc(sb + j * (UMMA_K * 128), BOX_MN_BYTES, 1024)
                                     : smem_desc(sb + j * (UMMA_K * 2), 16, 1024);
            umma_bf16(tmem_d, ad, bd, IDESC, (kb > kb0 || j > 0) ? 1u : 0u);
          }
          umma_commit(&empty[stage]);                 // frees the smem stage when these MMAs retire
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        umma_commit(&tfull[acc]);                     // accumulator complete -> epilogue
        acc ^= 1;
        if (acc == 0) acc_phase ^= 1;
      }
    }
  } else {
    const int q = warp & 3;                           // TMEM lane quarter this warp may access
    uint32_t acc = 0, acc_phase = 0;
    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
      const int tile = item / p.splits;
      const int m0 = (tile % p.tiles_m) * BLOCK_M, n0 = (tile / p.tiles_m) * BLOCK_N;
      mbar_wait(&tfull[acc], acc_phase);
      tc_fence_after();
      const int row = m0 + q * 32 + lane;
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + acc * BLOCK_N;
#pragma unroll 1
      for (int c = 0; c < BLOCK_N; c += 32) {
        if (n0 + c >= p.N) break;                     // warp-uniform
        uint32_t r[32];
        tmem_ld32(taddr + c, r);
        if (row < p.M) {
          const int col = n0 + c;
          if (ACCUM) {
            float* dst = reinterpret_cast<float*>(p.C) + (size_t)row * p.ldc + col;
#pragma unroll
            for (int j = 0; j < 32; j += 4) {
              if (col + j + 4 <= p.N) {
                asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst + j),
                             "f"(__uint_as_float(r[j])), "f"(__uint_as_float(r[j + 1])),
                             "f"(__uint_as_float(r[j + 2])), "f"(__uint_as_float(r[j + 3]))
                             : "memory");
              } else {
                for (int t = 0; t < 4; ++t)
                  if (col + j + t < p.N) atomicAdd(dst + j + t, __uint_as_float(r[j + t]));
              }
            }
          } else {
            bf16* dst = reinterpret_cast<bf16*>(p.C) + (size_t)row * p.ldc + col;
#pragma unroll
            for (int j = 0; j < 32; j += 8) {
              float v[8];
#pragma unroll
              for (int t = 0; t < 8; ++t) v[t] = __uint_as_float(r[j + t]);
              if (col + j + 8 <= p.N) {
                if (p.bias != nullptr) {
                  const float4 b0 = __ldg(reinterpret_cast<const float4*>(p.bias + col + j));
                  const float4 b1 = __ldg(reinterpret_cast<const float4*>(p.bias + col + j + 4));
                  v[0] += b0.x; v[1] += b0.y; v[2] += b0.z; v[3] += b0.w;
                  v[4] += b1.x; v[5] += b1.y; v[6] += b1.z; v[7] += b1.w;
                }
                store_vec<bf16>(dst + j, v);
              } else {
                for (int t = 0; t < 8; ++t)
                  if (col + j + t < p.N)
                    dst[j + t] = __float2bfloat16_rn(v[t] + (p.bias != nullptr ? p.bias[col + j + t] : 0.f));
              }
            }
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&tempty[acc]);
      acc ^= 1;
      if (acc == 0) acc_phase ^= 1;
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(TMEM_COLS) : "memory");
  }
}

// ------------------------------------------------------------------ host: tensor maps
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  static std::once_flag once;
  std::call_once(once, [] {
    void* f = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)f;
  });
  return fn;
}

struct MapKey {
  const void* ptr; uint64_t d0, d1, ld; uint32_t b0, b1;
  bool operator==(const MapKey& o) const {
    return ptr == o.ptr && d0 == o.d0 && d1 == o.d1 && ld == o.ld && b0 == o.b0 && b1 == o.b1;
  }
};
struct MapKeyHash {
  size_t operator()(const MapKey& k) const {
    size_t h = (size_t)k.ptr;
    for (uint64_t v : {k.d0, k.d1, k.ld, (uint64_t)k.b0, (uint64_t)k.b1}) h = h * 1000003u ^ (size_t)v;
    return h;
  }
};

// 2D bf16 tensor: dim0 (contiguous) extent d0, dim1 extent d1 with row stride ld elements; box {b0, b1}.
int make_map(CUtensorMap* out, const void* ptr, uint64_t d0, uint64_t d1, uint64_t ld, uint32_t b0, uint32_t b1) {
  static std::unordered_map<MapKey, CUtensorMap, MapKeyHash> cache;
  static std::mutex mu;
  MapKey key{ptr, d0, d1, ld, b0, b1};
  {
    std::lock_guard<std::mutex> g(mu);
    auto it = cache.find(key);
    if (it != cache.end()) { *out = it->second; return PACI_OK; }
  }
  EncodeTiledFn fn = encode_fn();
  if (!fn) return fail(PACI_ECUDA, "cuTensorMapEncodeTiled is not available from the driver");
  if ((uintptr_t)ptr % 16 || (ld * 2) % 16) return fail(PACI_EINVAL, "tcgen05 GEMM: operand not 16-byte aligned (ld=%llu)", (unsigned long long)ld);
  cuuint64_t dims[2] = {d0, d1};
  cuuint64_t strides[1] = {ld * 2};
  cuuint32_t box[2] = {b0, b1};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(ptr), dims, strides, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(PACI_ECUDA, "cuTensorMapEncodeTiled failed with %d", (int)r);
  std::lock_guard<std::mutex> g(mu);
  if (cache.size() > 4096) cache.clear();
  cache[key] = *out;
  return PACI_OK;
}

template <int BLOCK_N, bool A_MN, bool B_MN, bool ACCUM>
int launch(const CUtensorMap& tmA, const CUtensorMap& tmB, const Params& p, int grid, cudaStream_t s) {
  constexpr size_t SMEM = (size_t)STAGES * (BLOCK_M * BLOCK_K * 2 + BLOCK_N * BLOCK_K * 2) + 1024 + 256;
  auto kern = gemm_tc_kernel<BLOCK_N, A_MN, B_MN, ACCUM>;
  static bool attr_set = false;
  if (!attr_set) {
    PACI_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM));
    attr_set = true;
  }
  PACI_LAUNCH(kern, grid, NUM_THREADS, SMEM, s, tmA, tmB, p);
  return PACI_OK;
}

}  // namespace

int gemm_tc(int layout, int M, int N, int K, const void* A, int lda, const void* B, int ldb, const float* bias,
            void* C, int ldc, int out_f32_accum, cudaStream_t s) {
  if (M <= 0 || N <= 0) return PACI_OK;
  if (K <= 0) return fail(PACI_EINVAL, "tcgen05 GEMM: K=%d", K);
  if (layout < 0 || layout > 2) return fail(PACI_EINVAL, "gemm: layout %d", layout);
  if ((uintptr_t)C % 16 || (out_f32_accum ? ldc % 4 : ldc % 8))
    return fail(PACI_EINVAL, "tcgen05 GEMM: C not 16-byte aligned (ldc=%d)", ldc);
  if (bias != nullptr && (uintptr_t)bias % 16) return fail(PACI_EINVAL, "tcgen05 GEMM: bias not 16-byte aligned");
  const bool a_mn = layout == 2, b_mn = layout != 0;
  const int BN = N <= 128 ? 128 : 256;
  CUtensorMap tmA, tmB;
  int rc;
  // A: K-major [M rows][K contiguous] -> dims {K, M}, box {64, 128};  MN-major [K rows][M contiguous] -> {M, K}, {64, 64}
  rc = a_mn ? make_map(&tmA, A, M, K, lda, 64, BLOCK_K) : make_map(&tmA, A, K, M, lda, BLOCK_K, BLOCK_M);
  if (rc) return rc;
  rc = b_mn ? make_map(&tmB, B, N, K, ldb, 64, BLOCK_K) : make_map(&tmB, B, K, N, ldb, BLOCK_K, BN);
  if (rc) return rc;
  Params p;
  p.M = M; p.N = N; p.K = K; p.ldc = ldc; p.bias = bias; p.C = C;
  p.tiles_m = ceil_div(M, BLOCK_M);
  p.tiles_n = ceil_div(N, BN);
  p.kb_total = ceil_div(K, BLOCK_K);
  const int tiles = p.tiles_m * p.tiles_n, sms = num_sms();
  int splits = 1;
  if (out_f32_accum) {   // split-K over the contraction (tokens): partials meet in the fp32 red.add epilogue
    splits = std::max(1, std::min({ceil_div(2 * sms, tiles), p.kb_total / 4, 32}));
    const int kb_per = ceil_div(p.kb_total, splits);
    splits = ceil_div(p.kb_total, kb_per);            // every split owns at least one k-block
  }
  p.splits = splits;
  const int grid = std::min(tiles * splits, sms);
#define GO(BN_, AMN, BMN, ACC) return launch<BN_, AMN, BMN, ACC>(tmA, tmB, p, grid, s)
  if (BN == 128) {
    if (out_f32_accum) { if (layout == 0) GO(128, false, false, true); if (layout == 1) GO(128, false, true, true); GO(128, true, true, true); }
    if (layout == 0) GO(128, false, false, false); if (layout == 1) GO(128, false, true, false); GO(128, true, true, false);
  }
  if (out_f32_accum) { if (layout == 0) GO(256, false, false, true); if (layout == 1) GO(256, false, true, true); GO(256, true, true, true); }
  if (layout == 0) GO(256, false, false, false); if (layout == 1) GO(256, false, true, false); GO(256, true, true, false);
#undef GO
}

}  // namespace paci
