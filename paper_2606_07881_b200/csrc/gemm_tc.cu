// gemm_tc.cu -- bf16 GEMM on the 5th-generation tensor cores (tcgen05.mma), hand-written for sm_100a.
// Rows a3, a5, a7, a9, a10 (forward, "NT"), a12/a13 (dgrad with the CURRENT weights, "NN") and a14
// (wgrad whose epilogue ADDS into the fp32 accumulator G, "TN", split-K over tokens) of SURVEY.md 8(a).
//
// Structure: persistent, one CTA per SM, 192 threads; by default the two CTAs of a cluster (one TPC) work as a
// PAIR on a 256 x 256 tile (tcgen05.mma.cta_group::2, M = 256): each CTA stages its own 128 rows of A and HALF of
// the B tile, the leader issues the MMAs for both, each CTA keeps its 128 accumulator rows in its own TMEM.
//   warp 0      TMA producer: cp.async.bulk.tensor 2D tiles -> 128B-swizzled shared memory, 5-stage ring; in pair
//               mode both CTAs' bytes are counted on the LEADER's "full" mbarrier
//   warp 1      MMA issuer (leader CTA only): one thread issues tcgen05.mma (N = BLOCK_N, K = 16) from shared-
//               memory matrix descriptors; accumulators live in TMEM (2 buffers x BLOCK_N fp32 columns), so the
//               epilogue of tile i overlaps the main loop of tile i+1; tcgen05.commit (multicast to both CTAs)
//               frees a stage / publishes an accumulator
//   warps 2-5   epilogue: tcgen05.ld (32 lanes x 64 columns per warp and chunk) -> (+bias from registers, ->bf16)
//               -> 128B-swizzled staging box in shared memory -> TMA store, or, for the fp32 accumulator G
//               (beta = 1, Alg. 1 line 13), TMA reduce-add (cp.reduce.async.bulk.tensor .add): wgrad accumulation
//               and split-K partials are the same mechanism and need no separate kernel
// Pipelines: full/empty mbarriers between TMA and MMA, tmem_full / tmem_empty between MMA and epilogue (the
// peer's epilogue warps arrive on the leader's barrier through the cluster address space).
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
#include <cstdlib>
#include <mutex>
#include <unordered_map>

#include "common.cuh"
#include "tc_ptx.cuh"

namespace paci {

namespace {

constexpr int BLOCK_M = 128;
constexpr int BLOCK_K = 64;
constexpr int UMMA_K = 16;
constexpr int NUM_THREADS = 192;
constexpr int EPI_BUFS = 3;                 // staging boxes per epilogue warp: a box is reused only after the TMA store
                                            // issued EPI_BUFS chunks ago has read it (2 buffers left ~0.7 us of store
                                            // latency exposed per chunk: 3.1 us of epilogue for the last tile of a launch)
constexpr uint32_t EPI_STAGING_BYTES = 4 * EPI_BUFS * 4096;

using namespace tc;

struct Params {
  int M, N, K, ldc;
  int tiles_m, tiles_n, splits, kb_total;
  int range_mode;                                   // 1: workers own contiguous ranges of (tile, k-block) units
  const float* bias;
  void* C;
  int gelu;       // !ACCUM only: also store gelu(C) through tmC2 (MLP-up: the pre-activation is stashed, rows a7 + a8)
};

// ------------------------------------------------------------------ the kernel
// CG = 1: one CTA per tile of 128 x BLOCK_N.  CG = 2: a CTA pair (cluster of 2, same TPC) per tile of
// 256 x BLOCK_N: CTA r owns rows m0 + 128 r .. of A and of the accumulator, and stages columns
// n0 + r BLOCK_N/2 .. of B; the leader (rank 0) issues tcgen05.mma.cta_group::2 for both.
template <int CG, int BLOCK_N, int STAGES, bool A_MN, bool B_MN, bool ACCUM>
__global__ void __launch_bounds__(NUM_THREADS, 1)
gemm_tc_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
               const __grid_constant__ CUtensorMap tmC, const __grid_constant__ CUtensorMap tmC2, const Params p) {
  constexpr int BN_CTA = BLOCK_N / CG;                  // B rows staged by one CTA
  constexpr uint32_t A_BYTES = BLOCK_M * BLOCK_K * 2, B_BYTES = BN_CTA * BLOCK_K * 2;
  constexpr uint32_t STAGE_BYTES = A_BYTES + B_BYTES;
  constexpr uint32_t BOX_MN_BYTES = 64 * BLOCK_K * 2;   // one {64 mn, 64 k} box of an MN-major operand
  constexpr uint32_t TMEM_COLS = 2 * BLOCK_N;
  // instruction descriptor: D fp32 (bit 4), A/B bf16 (bits 7, 10), majors (15, 16), N>>3 at 17, M>>4 at 24
  constexpr uint32_t IDESC = (1u << 4) | (1u << 7) | (1u << 10) | ((A_MN ? 1u : 0u) << 15) |
                             ((B_MN ? 1u : 0u) << 16) | ((uint32_t)(BLOCK_N >> 3) << 17) |
                             ((uint32_t)((BLOCK_M * CG) >> 4) << 24);

  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  uint8_t* staging = smem + STAGES * STAGE_BYTES;        // 4 epilogue warps x EPI_BUFS buffers x 4 KB (1024-aligned)
  float* bias_s = (float*)(staging + EPI_STAGING_BYTES); // 4 epilogue warps x BLOCK_N floats
  uint64_t* full = (uint64_t*)(bias_s + 4 * BLOCK_N);
  uint64_t* empty = full + STAGES;
  uint64_t* tfull = empty + STAGES;
  uint64_t* tempty = tfull + 2;
  uint32_t* tmem_slot = (uint32_t*)(tempty + 2);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = CG == 2 ? cluster_ctarank() : 0u;
  const bool leader = rank == 0;

  if (threadIdx.x == 0) {
    for (int i = 0; i < STAGES; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&tfull[i], 1); mbar_init(&tempty[i], 4 * CG); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  // CTA pair: tcgen05.alloc.cta_group::2 must not be issued before the peer CTA is known to be running.  Without
  // this first cluster barrier the odd CTA's alloc blocked for ever, once in ~100 launches, whenever another
  // stream's multi-wave kernel shared the SMs (all other CTAs of the launch had finished; peer stuck in the second
  // barrier).  The second barrier makes both allocations (and both CTAs' mbarriers) exist before the leader's
  // first MMA writes the peer's TMEM.
  if (CG == 2) { __syncthreads(); cluster_sync_all(); }
  if (warp == 1) {
    if (CG == 2) {
      asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)),
                   "r"(TMEM_COLS) : "memory");
    } else {
      asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)),
                   "r"(TMEM_COLS) : "memory");
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
  }
  tc_fence_before();
  __syncthreads();
  if (CG == 2) {
    cluster_sync_all();
    if (warp == 1) asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
  }
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  const int n_items = p.tiles_m * p.tiles_n * p.splits;
  const int kb_per = (p.kb_total + p.splits - 1) / p.splits;
  const int worker = CG == 2 ? (int)(blockIdx.x >> 1) : (int)blockIdx.x;
  const int n_workers = CG == 2 ? (int)(gridDim.x >> 1) : (int)gridDim.x;
  // The work list of this CTA (pair), walked identically by the producer, the MMA issuer and the epilogue warps.
  // Item mode: items = tile x split, dealt round-robin.  Range mode (fp32 reduce-add output only): the (tile,
  // k-block) space is cut into n_workers equal contiguous ranges, so every worker does the same number of k-blocks
  // and flushes its accumulator wherever its range crosses a tile boundary (partials meet in the L2 adders).
  struct Work {
    long cur, end;
    int item, n_items, step, splits, kb_per, kb_total, range;
    __device__ __forceinline__ bool next(int& tile, int& kb0, int& kb1) {
      if (range) {
        if (cur >= end) return false;
        tile = (int)(cur / kb_total);
        kb0 = (int)(cur % kb_total);
        kb1 = (int)min((long)kb_total, kb0 + (end - cur));
        cur += kb1 - kb0;
        return true;
      }
      if (item >= n_items) return false;
      tile = item / splits;
      kb0 = (item % splits) * kb_per;
      kb1 = min(kb0 + kb_per, kb_total);
      item += step;
      return true;
    }
  };
  const long units = (long)p.tiles_m * p.tiles_n * p.kb_total;
  const Work work0{units * worker / n_workers, units * (worker + 1) / n_workers, worker, n_items, n_workers, p.splits, kb_per,
                   p.kb_total, p.range_mode};

  if (warp == 0) {
    if (lane == 0) {
      asm volatile("prefetch.tensormap [%0];" ::"l"(&tmA) : "memory");
      asm volatile("prefetch.tensormap [%0];" ::"l"(&tmB) : "memory");
      uint32_t stage = 0, phase = 0;
      Work work = work0;
      for (int tile, kb0, kb1; work.next(tile, kb0, kb1);) {
        const int m0 = (tile % p.tiles_m) * (BLOCK_M * CG) + (int)rank * BLOCK_M;
        const int n0 = (tile / p.tiles_m) * BLOCK_N + (int)rank * BN_CTA;
        for (int kb = kb0; kb < kb1; ++kb) {
          mbar_wait(&empty[stage], phase ^ 1, 1);
          uint8_t* sa = smem + stage * STAGE_BYTES;
          uint8_t* sb = sa + A_BYTES;
          const int k0 = kb * BLOCK_K;
          if (CG == 2) {
            // both CTAs' bytes are counted on the leader's barrier; its single arrival is this expect_tx
            if (leader) mbar_expect_tx(&full[stage], 2 * STAGE_BYTES);
            const uint32_t bar = mapa_rank(smem_u32(&full[stage]), 0);
            if (A_MN) {
#pragma unroll
              for (int i = 0; i < BLOCK_M / 64; ++i) tma_load_2d_pair(sa + i * BOX_MN_BYTES, &tmA, bar, m0 + i * 64, k0);
            } else {
              tma_load_2d_pair(sa, &tmA, bar, k0, m0);
            }
            if (B_MN) {
#pragma unroll
              for (int i = 0; i < BN_CTA / 64; ++i) tma_load_2d_pair(sb + i * BOX_MN_BYTES, &tmB, bar, n0 + i * 64, k0);
            } else {
              tma_load_2d_pair(sb, &tmB, bar, k0, n0);
            }
          } else {
            mbar_expect_tx(&full[stage], STAGE_BYTES);
            if (A_MN) {
#pragma unroll
              for (int i = 0; i < BLOCK_M / 64; ++i) tma_load_2d(sa + i * BOX_MN_BYTES, &tmA, &full[stage], m0 + i * 64, k0);
            } else {
              tma_load_2d(sa, &tmA, &full[stage], k0, m0);
            }
            if (B_MN) {
#pragma unroll
              for (int i = 0; i < BN_CTA / 64; ++i) tma_load_2d(sb + i * BOX_MN_BYTES, &tmB, &full[stage], n0 + i * 64, k0);
            } else {
              tma_load_2d(sb, &tmB, &full[stage], k0, n0);
            }
          }
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    if (lane == 0 && leader) {
      uint32_t stage = 0, phase = 0, acc = 0, acc_phase = 0;
      Work work = work0;
      for (int tile, kb0, kb1; work.next(tile, kb0, kb1);) {
        mbar_wait(&tempty[acc], acc_phase ^ 1, 2);      // epilogue (of both CTAs) has drained this accumulator
        tc_fence_after();
        const uint32_t tmem_d = tmem_base + acc * BLOCK_N;
        for (int kb = kb0; kb < kb1; ++kb) {
          mbar_wait(&full[stage], phase, 3);
          tc_fence_after();
          const uint32_t sa = smem_u32(smem + stage * STAGE_BYTES), sb = sa + A_BYTES;
#pragma unroll
          for (int j = 0; j < BLOCK_K / UMMA_K; ++j) {
            const uint64_t ad = A_MN ? smem_desc(sa + j * (UMMA_K * 128), BOX_MN_BYTES, 1024)
                                     : smem_desc(sa + j * (UMMA_K * 2), 16, 1024);
            const uint64_t bd = B_MN ? smem_desc(sb + j * (UMMA_K * 128), BOX_MN_BYTES, 1024)
                                     : smem_desc(sb + j * (UMMA_K * 2), 16, 1024);
            if (CG == 2) umma_bf16_pair(tmem_d, ad, bd, IDESC, (kb > kb0 || j > 0) ? 1u : 0u);
            else umma_bf16(tmem_d, ad, bd, IDESC, (kb > kb0 || j > 0) ? 1u : 0u);
          }
          if (CG == 2) umma_commit_pair(&empty[stage]); else umma_commit(&empty[stage]);   // frees the stage
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        if (CG == 2) umma_commit_pair(&tfull[acc]); else umma_commit(&tfull[acc]);         // -> epilogue
        acc ^= 1;
        if (acc == 0) acc_phase ^= 1;
      }
    }
  } else {
    // ===== epilogue warps: TMEM -> registers -> swizzled smem -> TMA store / TMA reduce-add =====
    // Warp w (TMEM lane quarter q = w & 3) owns 32 rows of the tile and a private pair of 4 KB staging
    // buffers, so the four warps never synchronise with each other.  One TMA box = 32 rows x 128 bytes
    // (64 bf16 or 32 fp32 columns), SWIZZLE_128B: 16-byte chunk c of row r sits at chunk c ^ (r & 7),
    // which makes the row-per-thread st.shared.v4 conflict-free.  TMA clips the box at the tensor edge.
    const int q = warp & 3;
    constexpr int CHUNK = ACCUM ? 32 : 64;            // columns per TMA box
    uint8_t* my_stage = staging + (warp - 2) * (EPI_BUFS * 4096);
    float* my_bias = bias_s + (warp - 2) * BLOCK_N;
    uint32_t acc = 0, acc_phase = 0, sbuf = 0;
    Work work = work0;
    for (int tile, kb0, kb1; work.next(tile, kb0, kb1);) {
      const int m0 = (tile % p.tiles_m) * (BLOCK_M * CG) + (int)rank * BLOCK_M, n0 = (tile / p.tiles_m) * BLOCK_N;
      if (!ACCUM) {                                   // bias slice of this tile, fetched under the main loop
#pragma unroll
        for (int i = 0; i < BLOCK_N / 32; ++i) {
          const int col = n0 + i * 32 + lane;
          my_bias[i * 32 + lane] = (p.bias != nullptr && col < p.N) ? __ldg(p.bias + col) : 0.f;
        }
        __syncwarp();
      }
      mbar_wait_many(&tfull[acc], acc_phase, 4);     // 128 threads wait a whole main loop: sleep between polls
      tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + acc * BLOCK_N;
#pragma unroll 1
      for (int c = 0; c < BLOCK_N; c += CHUNK) {
        if (n0 + c >= p.N) break;                     // warp-uniform
        const bool gelu = !ACCUM && p.gelu != 0;       // kernel-uniform
        uint8_t* buf = gelu ? my_stage : my_stage + sbuf * 4096;
        uint8_t* buf2 = my_stage + 4096;               // gelu: second output tile of the same chunk
        if (!gelu) sbuf = sbuf + 1 == EPI_BUFS ? 0 : sbuf + 1;
        if (lane == 0) { if (gelu) bulk_wait_read<0>(); else bulk_wait_read<EPI_BUFS - 1>(); }   // staging buffer(s) free again
        __syncwarp();
        uint8_t* rowp = buf + lane * 128;
        if (ACCUM) {
          uint32_t r[32];
          tmem_ld32(taddr + c, r);
#pragma unroll
          for (int i = 0; i < 8; ++i)
            sts128(rowp + ((i ^ (lane & 7)) << 4), r[4 * i], r[4 * i + 1], r[4 * i + 2], r[4 * i + 3]);
        } else {
          uint32_t r64[64];                            // both halves of the chunk in flight before one wait
          tmem_ld32_nowait(taddr + c, r64);
          tmem_ld32_nowait(taddr + c + 32, r64 + 32);
          // the chunk's 64 bias values go to registers up front: interleaved with the (volatile, memory-
          // clobbering) st.shared they serialised into 8 load -> add -> store chains, 0.4 us per chunk
          float4 bq[16];
#pragma unroll
          for (int k = 0; k < 16; ++k) bq[k] = *reinterpret_cast<const float4*>(my_bias + c + 4 * k);
          tmem_ld_wait();
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            const uint32_t* r = r64 + 32 * h;
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const float4 b0 = bq[8 * h + 2 * i];
              const float4 b1 = bq[8 * h + 2 * i + 1];
              uint32_t w[4];
              w[0] = pack_bf16x2(__uint_as_float(r[8 * i]) + b0.x, __uint_as_float(r[8 * i + 1]) + b0.y);
              w[1] = pack_bf16x2(__uint_as_float(r[8 * i + 2]) + b0.z, __uint_as_float(r[8 * i + 3]) + b0.w);
              w[2] = pack_bf16x2(__uint_as_float(r[8 * i + 4]) + b1.x, __uint_as_float(r[8 * i + 5]) + b1.y);
              w[3] = pack_bf16x2(__uint_as_float(r[8 * i + 6]) + b1.z, __uint_as_float(r[8 * i + 7]) + b1.w);
              const uint32_t off = (uint32_t)(((4 * h + i) ^ (lane & 7)) << 4);
              sts128(rowp + off, w[0], w[1], w[2], w[3]);
              if (gelu) {                              // gelu of the ROUNDED pre-activation, as backward will see it
                uint32_t gw[4];
#pragma unroll
                for (int u = 0; u < 4; ++u)
                  gw[u] = pack_bf16x2(gelu_bf16(__uint_as_float(w[u] << 16)), gelu_bf16(__uint_as_float(w[u] & 0xffff0000u)));
                sts128(buf2 + lane * 128 + off, gw[0], gw[1], gw[2], gw[3]);
              }
            }
          }
        }
        fence_async_smem();                           // generic-proxy writes -> visible to the TMA engine
        __syncwarp();
        if (lane == 0) {
          if (ACCUM) tma_reduce_add_2d(&tmC, buf, n0 + c, m0 + q * 32);
          else tma_store_2d(&tmC, buf, n0 + c, m0 + q * 32);
          if (gelu) tma_store_2d(&tmC2, buf2, n0 + c, m0 + q * 32);
          bulk_commit();
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        if (CG == 2) mbar_arrive_cluster(mapa_rank(smem_u32(&tempty[acc]), 0));
        else mbar_arrive(&tempty[acc]);
      }
      acc ^= 1;
      if (acc == 0) acc_phase ^= 1;
    }
    if (lane == 0) bulk_wait_read<0>();               // smem must outlive the last TMA read; the global writes are
                                                      // complete at kernel end like any other store
  }
  tc_fence_before();
  __syncthreads();
  if (CG == 2) cluster_sync_all();                     // no CTA leaves while its pair can still signal it
  if (warp == 1) {
    tc_fence_after();
    if (CG == 2)
      asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(TMEM_COLS) : "memory");
    else
      asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(TMEM_COLS) : "memory");
  }
  if (CG == 2) cluster_sync_all();                     // pair-wide dealloc: neither CTA exits before both freed
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
  const void* ptr; uint64_t d0, d1, ld; uint32_t b0, b1, esz;
  bool operator==(const MapKey& o) const {
    return ptr == o.ptr && d0 == o.d0 && d1 == o.d1 && ld == o.ld && b0 == o.b0 && b1 == o.b1 && esz == o.esz;
  }
};
struct MapKeyHash {
  size_t operator()(const MapKey& k) const {
    size_t h = (size_t)k.ptr;
    for (uint64_t v : {k.d0, k.d1, k.ld, (uint64_t)k.b0, (uint64_t)k.b1, (uint64_t)k.esz}) h = h * 1000003u ^ (size_t)v;
    return h;
  }
};

// 2D tensor of bf16 (esz 2) or fp32 (esz 4): dim0 (contiguous) extent d0, dim1 extent d1 with row stride ld
// elements; box {b0, b1}; 128-byte swizzle.
int make_map(CUtensorMap* out, const void* ptr, uint64_t d0, uint64_t d1, uint64_t ld, uint32_t b0, uint32_t b1,
             uint32_t esz = 2) {
  static std::unordered_map<MapKey, CUtensorMap, MapKeyHash> cache;
  static std::mutex mu;
  MapKey key{ptr, d0, d1, ld, b0, b1, esz};
  {
    std::lock_guard<std::mutex> g(mu);
    auto it = cache.find(key);
    if (it != cache.end()) { *out = it->second; return PACI_OK; }
  }
  EncodeTiledFn fn = encode_fn();
  if (!fn) return fail(PACI_ECUDA, "cuTensorMapEncodeTiled is not available from the driver");
  if ((uintptr_t)ptr % 16 || (ld * esz) % 16) return fail(PACI_EINVAL, "tcgen05 GEMM: operand not 16-byte aligned (ld=%llu)", (unsigned long long)ld);
  cuuint64_t dims[2] = {d0, d1};
  cuuint64_t strides[1] = {ld * esz};
  cuuint32_t box[2] = {b0, b1};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = fn(out, esz == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(ptr), dims, strides, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(PACI_ECUDA, "cuTensorMapEncodeTiled failed with %d", (int)r);
  std::lock_guard<std::mutex> g(mu);
  if (cache.size() > 4096) cache.clear();
  cache[key] = *out;
  return PACI_OK;
}


template <int CG, int BLOCK_N, int STAGES, bool A_MN, bool B_MN, bool ACCUM>
int launch(const CUtensorMap& tmA, const CUtensorMap& tmB, const CUtensorMap& tmC, const CUtensorMap& tmC2,
           const Params& p, int grid, cudaStream_t s) {
  constexpr size_t SMEM = (size_t)STAGES * (BLOCK_M * BLOCK_K * 2 + (BLOCK_N / CG) * BLOCK_K * 2) +
                          EPI_STAGING_BYTES + 4 * BLOCK_N * 4 + 1024 + 256;
  static_assert(SMEM <= 232448, "shared memory budget of one sm_100 CTA");
  auto kern = gemm_tc_kernel<CG, BLOCK_N, STAGES, A_MN, B_MN, ACCUM>;
  { int rc_ = set_max_dynamic_smem((const void*)kern, (int)SMEM); if (rc_) return rc_; }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(NUM_THREADS);
  cfg.dynamicSmemBytes = SMEM;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = CG;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  PACI_CUDA_OK(cudaLaunchKernelEx(&cfg, kern, tmA, tmB, tmC, tmC2, p));
  g_launches.fetch_add(1, std::memory_order_relaxed);
  return PACI_OK;
}

thread_local int32_t g_last_plan[6] = {0, 0, 0, 0, 0, 0};

}  // namespace

int make_tensor_map(CUtensorMap* out, const void* ptr, uint64_t d0, uint64_t d1, uint64_t ld, uint32_t b0,
                    uint32_t b1, uint32_t esz) {
  return make_map(out, ptr, d0, d1, ld, b0, b1, esz);
}

int gemm_tc(int layout, int M, int N, int K, const void* A, int lda, const void* B, int ldb, const float* bias,
            void* C, int ldc, int out_f32_accum, cudaStream_t s, void* gelu_out) {
  if (M <= 0 || N <= 0) return PACI_OK;
  if (gelu_out != nullptr && (out_f32_accum || (uintptr_t)gelu_out % 16))
    return fail(PACI_EINVAL, "tcgen05 GEMM: gelu output needs the bf16 epilogue and a 16-byte aligned pointer");
  if (K <= 0) return fail(PACI_EINVAL, "tcgen05 GEMM: K=%d", K);
  if (layout < 0 || layout > 2) return fail(PACI_EINVAL, "gemm: layout %d", layout);
  if ((uintptr_t)C % 16 || (out_f32_accum ? ldc % 4 : ldc % 8))
    return fail(PACI_EINVAL, "tcgen05 GEMM: C not 16-byte aligned (ldc=%d)", ldc);
  if (bias != nullptr && (uintptr_t)bias % 16) return fail(PACI_EINVAL, "tcgen05 GEMM: bias not 16-byte aligned");
  const bool a_mn = layout == 2, b_mn = layout != 0;
  constexpr int CG = 2;                              // CTA pair (cluster of 2, one TPC) per 256-row tile
  const int BN = N <= 128 ? 128 : 256;
  CUtensorMap tmA, tmB, tmC, tmC2;
  int rc;
  // A: K-major [M rows][K contiguous] -> dims {K, M}, box {64, 128};  MN-major [K rows][M contiguous] -> {M, K}, {64, 64}
  rc = a_mn ? make_map(&tmA, A, M, K, lda, 64, BLOCK_K) : make_map(&tmA, A, K, M, lda, BLOCK_K, BLOCK_M);
  if (rc) return rc;
  rc = b_mn ? make_map(&tmB, B, N, K, ldb, 64, BLOCK_K) : make_map(&tmB, B, K, N, ldb, BLOCK_K, BN / CG);
  if (rc) return rc;
  // C: box of 32 rows x 128 bytes, written by one epilogue warp per TMA store / reduce-add
  rc = out_f32_accum ? make_map(&tmC, C, N, M, ldc, 32, 32, 4) : make_map(&tmC, C, N, M, ldc, 64, 32, 2);
  if (rc) return rc;
  tmC2 = tmC;
  if (gelu_out != nullptr && (rc = make_map(&tmC2, gelu_out, N, M, ldc, 64, 32, 2))) return rc;
  Params p;
  p.M = M; p.N = N; p.K = K; p.ldc = ldc; p.bias = bias; p.C = C; p.gelu = gelu_out != nullptr;
  p.tiles_m = ceil_div(M, BLOCK_M * CG);
  p.tiles_n = ceil_div(N, BN);
  p.kb_total = ceil_div(K, BLOCK_K);
  const int tiles = p.tiles_m * p.tiles_n, workers = std::max(1, num_sms() / CG);
  int splits = 1;
  if (out_f32_accum) {
    // split-K over the contraction (tokens): partials meet in the fp32 TMA reduce-add epilogue.  Cost model in
    // k-block units: rounds of the persistent grid x (k-blocks per item + EPI), where EPI ~ 8 k-blocks stands
    // for an item's reduce-add epilogue (every extra split re-sends the whole fp32 tile through the L2 adders:
    // 8 splits of the 4096x1024 wgrad measured 73 us against 1 split's 1.73-round quantisation loss).
    const int max_s = std::max(1, std::min(p.kb_total / 4, 32));
    const int EPI = 8;
    long best = -1;
    for (int sp = 1; sp <= max_s; ++sp) {
      const int kb_per = ceil_div(p.kb_total, sp);
      if (ceil_div(p.kb_total, kb_per) != sp) continue;        // every split owns at least one k-block
      const long rounds = ceil_div((long)tiles * sp, workers);
      const long cost = rounds * (kb_per + EPI);
      if (best < 0 || cost < best) { best = cost; splits = sp; }
    }
  }
  p.splits = splits;
  p.range_mode = 0;
  if (out_f32_accum) {
    // equal contiguous (tile, k-block) ranges instead of whole items: U / W k-blocks per worker plus one flush per
    // tile boundary crossed (+1).  Taken for outputs of many rounds (the LM-head wgrad: 788 tiles, 10.65 rounds ->
    // 0.659 to 0.597 ms); with fewer tiles than two rounds the k-block rate itself drops when every pair is busy
    // and the round-robin splits measured the same or better
    const int EPI = 8;
    const long units = (long)tiles * p.kb_total;
    const long per = ceil_div(units, (long)workers);
    const long cost = per + (ceil_div(per, (long)p.kb_total) + 1) * EPI;
    const long item_cost = ceil_div((long)tiles * splits, (long)workers) * (ceil_div(p.kb_total, splits) + EPI);
    if (tiles >= 2 * workers && cost < item_cost) p.range_mode = 1;
  }
  // balanced persistent grid: the same number of rounds on the fewest workers (128 tiles on 74 pairs take 2
  // rounds; so do 64 pairs, and the other 20 SMs stay free for the other stage streams' kernels)
  const int items = tiles * splits;
  const int rounds = ceil_div(items, workers);
  const int grid = (p.range_mode ? workers : ceil_div(items, rounds)) * CG;
#define GO(CG_, BN_, ST_, AMN, BMN, ACC) return launch<CG_, BN_, ST_, AMN, BMN, ACC>(tmA, tmB, tmC, tmC2, p, grid, s)
#define BY_LAYOUT(CG_, BN_, ST_)                                                                          \
  do {                                                                                                    \
    if (out_f32_accum) {                                                                                  \
      if (layout == 0) GO(CG_, BN_, ST_, false, false, true);                                             \
      if (layout == 1) GO(CG_, BN_, ST_, false, true, true);                                              \
      GO(CG_, BN_, ST_, true, true, true);                                                                \
    }                                                                                                     \
    if (layout == 0) GO(CG_, BN_, ST_, false, false, false);                                              \
    if (layout == 1) GO(CG_, BN_, ST_, false, true, false);                                               \
    GO(CG_, BN_, ST_, true, true, false);                                                                 \
  } while (0)
  g_last_plan[0] = CG; g_last_plan[1] = BN; g_last_plan[2] = splits; g_last_plan[3] = p.range_mode;
  g_last_plan[4] = grid; g_last_plan[5] = tiles;
  if (BN == 128) BY_LAYOUT(2, 128, 7);
  BY_LAYOUT(2, 256, 5);
#undef BY_LAYOUT
#undef GO
}

void gemm_tc_last_plan(int32_t* out6) {
  for (int i = 0; i < 6; ++i) out6[i] = g_last_plan[i];
}

}  // namespace paci
