// gemm_tc.cu -- bf16 GEMM on the 5th-generation tensor cores (tcgen05.mma), hand-written for sm_100a.
// Rows a3, a5, a7, a9, a10 (forward, "NT"), a12/a13 (dgrad with the CURRENT weights, "NN") and a14
// (wgrad whose epilogue ADDS into the fp32 accumulator G, "TN", split-K over tokens) of SURVEY.md 8(a).
//
// Structure: persistent, one CTA per SM, 192 threads; by default the two CTAs of a cluster (one TPC) work as a
// PAIR on a 256 x 256 tile (tcgen05.mma.cta_group::2, M = 256): each CTA stages its own 128 rows of A and HALF of
// the B tile, the leader issues the MMAs for both, each CTA keeps its 128 accumulator rows in its own TMEM.
//   warp 4      TMA producer: cp.async.bulk.tensor 2D tiles -> 128B-swizzled shared memory, 5-stage ring; in pair
//               mode both CTAs' bytes are counted on the LEADER's "full" mbarrier
//   warp 5      MMA issuer (leader CTA only): one thread issues tcgen05.mma (N = BLOCK_N, K = 16) from shared-
//               memory matrix descriptors; accumulators live in TMEM (2 buffers x BLOCK_N fp32 columns), so the
//               epilogue of tile i overlaps the main loop of tile i+1; tcgen05.commit (multicast to both CTAs)
//               frees a stage / publishes an accumulator
//   warps 0-3   epilogue: tcgen05.ld (32 lanes x 64 columns per warp and chunk) -> (+bias from registers, ->bf16)
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
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <type_traits>
#include <vector>
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
constexpr float LOG2E_F = 1.4426950408889634f;
constexpr int EPI_BUFS = 4;                 // staging boxes per epilogue warp: a box is reused only after the TMA store
                                            // issued EPI_BUFS chunks ago has read it (2 buffers left ~0.7 us of store
                                            // latency exposed per chunk); the GELU epilogue uses them as two PAIRS
constexpr uint32_t EPI_STAGING_BYTES = 4 * EPI_BUFS * 4096;
constexpr int MAX_WORKERS = 80;             // CTA pairs of one launch (74 on a B200)
constexpr int MAX_PROB = 2;                 // problems per launch (a dgrad and the wgrad that shares its dy operand)

using namespace tc;

// One GEMM of a launch.  Layout and epilogue are RUNTIME properties, so one kernel serves NT / NN / TN, the bf16 store
// and the fp32 reduce-add epilogue, and two different problems can share one persistent grid.
struct Prob {
  int M, N, K;
  int tiles_m, tiles_n, kb_total;
  int splits;        // item mode: items = tile x split, dealt round-robin
  int range_mode;    // 1: worker w owns the contiguous (tile, k-block) units [ustart[w], ustart[w+1])   (accum only)
  int a_mn, b_mn;    // operand majors: 0 = K-major, 1 = MN-major
  int accum;         // 0: C is bf16, overwritten, + bias;  1: C is fp32 and the product is ADDED (TMA reduce-add)
  int gelu;          // !accum only: also store gelu(C) through the second map (MLP-up: rows a7 + a8)
  // !accum, !gelu, out-proj dgrad only (row a17's prologue): C is dO [mu T, H 64]; also emit delta[b,h,t] =
  // sum_d dO O over the 64 columns of head h (one epilogue chunk) and lse2 = lse log2(e)
  const void* dl_o;  // attention output O, bf16 [M, N] with row stride dl_ldo; NULL: no delta epilogue
  const float* dl_lse;
  float* dl_delta;
  float* dl_lse2;
  int dl_ldo, dl_T, dl_H;
  const float* bias;
};
struct Params {
  Prob pr[MAX_PROB];
  int n_prob;
  int ustart[MAX_PROB][MAX_WORKERS + 1];
};
struct Maps { CUtensorMap a[MAX_PROB], b[MAX_PROB], c[MAX_PROB], c2; };

// The work list of one CTA pair, walked identically by the producer, the MMA issuer and the epilogue warps: the
// problems in order; inside a problem either whole items (tile x split, round-robin) or the worker's contiguous range
// of (tile, k-block) units, cut wherever it crosses a tile boundary (partials meet in the L2 adders).
struct Work {
  int q, item;
  long cur, end;
  bool started;
  __device__ __forceinline__ Work() : q(0), item(0), cur(0), end(0), started(false) {}
  __device__ __forceinline__ bool next(const Params& p, int worker, int n_workers, int& tile, int& kb0, int& kb1) {
    while (q < p.n_prob) {
      const Prob& pr = p.pr[q];
      if (!started) {
        started = true;
        if (pr.range_mode) { cur = p.ustart[q][worker]; end = p.ustart[q][worker + 1]; }
        else item = worker;
      }
      if (pr.range_mode) {
        if (cur < end) {
          tile = (int)(cur / pr.kb_total);
          kb0 = (int)(cur % pr.kb_total);
          kb1 = (int)min((long)pr.kb_total, kb0 + (end - cur));
          cur += kb1 - kb0;
          return true;
        }
      } else {
        const int kb_per = (pr.kb_total + pr.splits - 1) / pr.splits;
        if (item < pr.tiles_m * pr.tiles_n * pr.splits) {
          tile = item / pr.splits;
          kb0 = (item % pr.splits) * kb_per;
          kb1 = min(kb0 + kb_per, pr.kb_total);
          item += n_workers;
          return true;
        }
      }
      ++q;
      started = false;
    }
    return false;
  }
};

// ------------------------------------------------------------------ the kernel
// A CTA pair (cluster of 2, same TPC) per tile of 256 x BLOCK_N: CTA r owns rows m0 + 128 r .. of A and of the
// accumulator, and stages columns n0 + r BLOCK_N/2 .. of B; the leader (rank 0) issues tcgen05.mma.cta_group::2 for both.
template <int BLOCK_N, int STAGES>
__global__ void __launch_bounds__(NUM_THREADS, 1)
gemm_tc_kernel(const __grid_constant__ Maps maps, const __grid_constant__ Params p) {
  constexpr int CG = 2;
  constexpr int BN_CTA = BLOCK_N / CG;                  // B rows staged by one CTA
  constexpr uint32_t A_BYTES = BLOCK_M * BLOCK_K * 2, B_BYTES = BN_CTA * BLOCK_K * 2;
  constexpr uint32_t STAGE_BYTES = A_BYTES + B_BYTES;
  constexpr uint32_t BOX_MN_BYTES = 64 * BLOCK_K * 2;   // one {64 mn, 64 k} box of an MN-major operand
  constexpr uint32_t TMEM_COLS = 2 * BLOCK_N;
  // instruction descriptor: D fp32 (bit 4), A/B bf16 (bits 7, 10), majors (15, 16), N>>3 at 17, M>>4 at 24
  constexpr uint32_t IDESC0 = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(BLOCK_N >> 3) << 17) |
                              ((uint32_t)((BLOCK_M * CG) >> 4) << 24);

  extern __shared__ __align__(1024) uint8_t smem[];     // 128B-swizzled tiles need 1024-byte alignment (checked below)
  uint8_t* staging = smem + STAGES * STAGE_BYTES;        // 4 epilogue warps x EPI_BUFS buffers x 4 KB
  float* bias_s = (float*)(staging + EPI_STAGING_BYTES); // 4 epilogue warps x 2 x 64 floats (chunk-wise, double-buffered)
  uint64_t* full = (uint64_t*)(bias_s + 4 * 128);
  uint64_t* empty = full + STAGES;
  uint64_t* tfull = empty + STAGES;
  uint64_t* tempty = tfull + 2;
  uint32_t* tmem_slot = (uint32_t*)(tempty + 2);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const bool leader = rank == 0;

  if ((smem_u32(smem) & 1023u) != 0) __trap();
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
  __syncthreads();
  cluster_sync_all();
  if (warp == 5)
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)),
                 "r"(TMEM_COLS) : "memory");
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();
  if (warp == 5) asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  if (threadIdx.x == 4 * 32) {                         // the descriptors are kernel parameters: fetch them before the wait
    for (int q = 0; q < p.n_prob; ++q) {
      asm volatile("prefetch.tensormap [%0];" ::"l"(&maps.a[q]) : "memory");
      asm volatile("prefetch.tensormap [%0];" ::"l"(&maps.b[q]) : "memory");
      asm volatile("prefetch.tensormap [%0];" ::"l"(&maps.c[q]) : "memory");
    }
  }
  PACI_PDL_SYNC;                                       // set-up above overlaps the previous kernel's tail

  const int worker = (int)(blockIdx.x >> 1);
  const int n_workers = (int)(gridDim.x >> 1);

  // Warp roles: epilogue = warps 0-3 (TMEM lane quarter = warp id), TMA producer = warp 4, MMA issuer = warp 5.  The
  // scheduler of an SM sub-partition prefers the highest warp id among its ready warps, so the two single-thread roles
  // that pace the main loop are never queued behind an epilogue warp of the same sub-partition.
  if (warp == 4) {
    if (lane == 0) {
      uint32_t stage = 0, phase = 0;
      const uint32_t full0 = mapa_rank(smem_u32(&full[0]), 0);     // the LEADER's full[0]; full[i] is 8 i bytes further
      const uint32_t smem0 = smem_u32(smem);
      Work work;
      for (int tile, kb0, kb1; work.next(p, worker, n_workers, tile, kb0, kb1);) {
        const Prob& pr = p.pr[work.q];
        const CUtensorMap* tmA = &maps.a[work.q];
        const CUtensorMap* tmB = &maps.b[work.q];
        const int m0 = (tile % pr.tiles_m) * (BLOCK_M * CG) + (int)rank * BLOCK_M;
        const int n0 = (tile / pr.tiles_m) * BLOCK_N + (int)rank * BN_CTA;
        // the k-block loop is specialised at compile time on the operand majors (a runtime layout flag inside it cost
        // 7-11% of the GEMM: measured); the dispatch is per work item
        auto kloop = [&](auto a_mn_t, auto b_mn_t) {
          constexpr bool a_mn = decltype(a_mn_t)::value, b_mn = decltype(b_mn_t)::value;
          for (int kb = kb0; kb < kb1; ++kb) {
            mbar_wait_lean(&empty[stage], phase ^ 1);
            const uint32_t sa = smem0 + stage * STAGE_BYTES, sb = sa + A_BYTES;
            const int k0 = kb * BLOCK_K;
            // both CTAs' bytes are counted on the leader's barrier; its single arrival is this expect_tx
            if (leader) mbar_expect_tx(&full[stage], 2 * STAGE_BYTES);
            const uint32_t bar = full0 + stage * 8;
            if (a_mn) {
#pragma unroll
              for (int i = 0; i < BLOCK_M / 64; ++i) tma_load_2d_pair_s(sa + i * BOX_MN_BYTES, tmA, bar, m0 + i * 64, k0);
            } else {
              tma_load_2d_pair_s(sa, tmA, bar, k0, m0);
            }
            if (b_mn) {
#pragma unroll
              for (int i = 0; i < BN_CTA / 64; ++i) tma_load_2d_pair_s(sb + i * BOX_MN_BYTES, tmB, bar, n0 + i * 64, k0);
            } else {
              tma_load_2d_pair_s(sb, tmB, bar, k0, n0);
            }
            if (++stage == STAGES) { stage = 0; phase ^= 1; }
          }
        };
        if (!pr.b_mn) kloop(std::false_type{}, std::false_type{});          // NT
        else if (!pr.a_mn) kloop(std::false_type{}, std::true_type{});      // NN
        else kloop(std::true_type{}, std::true_type{});                     // TN
      }
    }
  } else if (warp == 5) {
    if (lane == 0 && leader) {
      // The single issuing thread is on the critical path of every k-block (wait, fence, 4 MMAs, commit against 4 x 128
      // tensor cycles), so everything that does not change per MMA is hoisted: a shared-memory descriptor is a constant
      // per (problem, operand) plus the tile's address in 16-byte units, and a K = 16 step adds a constant to it.
      uint32_t stage = 0, phase = 0, acc = 0, acc_phase = 0;
      const uint32_t smem16 = smem_u32(smem) >> 4;
      Work work;
      for (int tile, kb0, kb1; work.next(p, worker, n_workers, tile, kb0, kb1);) {
        const Prob& pr = p.pr[work.q];
        mbar_wait_lean(&tempty[acc], acc_phase ^ 1);    // epilogue (of both CTAs) has drained this accumulator
        tc_fence_after();
        const uint32_t tmem_d = tmem_base + acc * BLOCK_N;
        auto kloop = [&](auto a_mn_t, auto b_mn_t) {
          constexpr bool a_mn = decltype(a_mn_t)::value, b_mn = decltype(b_mn_t)::value;
          constexpr uint32_t idesc = IDESC0 | ((a_mn ? 1u : 0u) << 15) | ((b_mn ? 1u : 0u) << 16);
          constexpr uint32_t a_step = (a_mn ? UMMA_K * 128 : UMMA_K * 2) >> 4, b_step = (b_mn ? UMMA_K * 128 : UMMA_K * 2) >> 4;
          const uint64_t adesc0 = a_mn ? smem_desc(0, BOX_MN_BYTES, 1024) : smem_desc(0, 16, 1024);
          const uint64_t bdesc0 = b_mn ? smem_desc(0, BOX_MN_BYTES, 1024) : smem_desc(0, 16, 1024);
          uint32_t accumulate = 0;
          for (int kb = kb0; kb < kb1; ++kb) {
            mbar_wait_lean(&full[stage], phase);
            tc_fence_after();
            const uint32_t sa16 = smem16 + stage * (STAGE_BYTES >> 4);
            uint64_t ad = adesc0 + sa16, bd = bdesc0 + (sa16 + (A_BYTES >> 4));
#pragma unroll
            for (int j = 0; j < BLOCK_K / UMMA_K; ++j) {
              umma_bf16_pair(tmem_d, ad, bd, idesc, accumulate);
              accumulate = 1;
              ad += a_step;
              bd += b_step;
            }
            umma_commit_pair(&empty[stage]);             // frees the stage
            if (++stage == STAGES) { stage = 0; phase ^= 1; }
          }
        };
        if (!pr.b_mn) kloop(std::false_type{}, std::false_type{});          // NT
        else if (!pr.a_mn) kloop(std::false_type{}, std::true_type{});      // NN
        else kloop(std::true_type{}, std::true_type{});                     // TN
        umma_commit_pair(&tfull[acc]);                   // -> epilogue
        acc ^= 1;
        if (acc == 0) acc_phase ^= 1;
      }
    }
  } else {
    // ===== epilogue warps: TMEM -> registers -> swizzled smem -> TMA store / TMA reduce-add =====
    // Warp w (TMEM lane quarter q = w & 3) owns 32 rows of the tile and EPI_BUFS private 4 KB staging buffers, so the
    // four warps never synchronise with each other.  One TMA box = 32 rows x 128 bytes (64 bf16 or 32 fp32 columns),
    // SWIZZLE_128B: 16-byte chunk c of row r sits at chunk c ^ (r & 7), which makes the row-per-thread st.shared.v4
    // conflict-free.  TMA clips the box at the tensor edge.
    const int q = warp & 3;
    uint8_t* my_stage = staging + warp * (EPI_BUFS * 4096);
    float* my_bias = bias_s + warp * 128;
    uint32_t acc = 0, acc_phase = 0, sbuf = 0;
    Work work;
    for (int tile, kb0, kb1; work.next(p, worker, n_workers, tile, kb0, kb1);) {
      const Prob& pr = p.pr[work.q];
      const CUtensorMap* tmC = &maps.c[work.q];
      const int m0 = (tile % pr.tiles_m) * (BLOCK_M * CG) + (int)rank * BLOCK_M, n0 = (tile / pr.tiles_m) * BLOCK_N;
      const bool accum = pr.accum != 0;
      // bias slice of this tile: lane l keeps columns l, l + 32, ... in registers (fetched under the main loop, so no
      // global-load latency sits inside the chunk loop) and hands them to shared memory one 64-column chunk ahead
      float breg[BLOCK_N / 32];
      if (!accum) {
        const float* bias = pr.bias;
        const int N = pr.N;
#pragma unroll
        for (int i = 0; i < BLOCK_N / 32; ++i) {
          const int col = n0 + i * 32 + lane;
          breg[i] = (bias != nullptr && col < N) ? __ldg(bias + col) : 0.f;
        }
        my_bias[lane] = breg[0];
        my_bias[32 + lane] = breg[1];
        __syncwarp();
      }
      mbar_wait_many(&tfull[acc], acc_phase, 4);     // 128 threads wait a whole main loop: sleep between polls
      tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + acc * BLOCK_N;
      if (accum) {
#pragma unroll 1
        for (int c = 0; c < BLOCK_N; c += 32) {
          if (n0 + c >= pr.N) break;                  // warp-uniform
          uint8_t* buf = my_stage + sbuf * 4096;
          sbuf = (sbuf + 1) % EPI_BUFS;
          if (lane == 0) bulk_wait_read<EPI_BUFS - 1>();   // this staging buffer is free again
          __syncwarp();
          uint8_t* rowp = buf + lane * 128;
          uint32_t r[32];
          tmem_ld32(taddr + c, r);
#pragma unroll
          for (int i = 0; i < 8; ++i)
            sts128(rowp + ((i ^ (lane & 7)) << 4), r[4 * i], r[4 * i + 1], r[4 * i + 2], r[4 * i + 3]);
          fence_async_smem();                         // generic-proxy writes -> visible to the TMA engine
          __syncwarp();
          if (lane == 0) {
            tma_reduce_add_2d(tmC, buf, n0 + c, m0 + q * 32);
            bulk_commit();
          }
        }
      } else {
        // specialised at compile time on the GELU output: as a runtime flag it put eight branch regions into every
        // chunk (one per 16-byte store), which kept the plain epilogue's 64 adds and 32 packs from overlapping
        auto chunks = [&](auto mode_t) {
        constexpr int mode = decltype(mode_t)::value;
        constexpr bool gelu = mode == 1, with_delta = mode == 2;
        // delta epilogue: thread = one row (b, t) of dO; a 64-column chunk is exactly one head
        const int drow = m0 + q * 32 + lane;
        const bool drow_ok = with_delta && drow < pr.M;
        const bf16* dl_orow = reinterpret_cast<const bf16*>(pr.dl_o) + (size_t)(drow_ok ? drow : 0) * pr.dl_ldo + n0;
        const int dl_b = with_delta ? drow / pr.dl_T : 0, dl_t = with_delta ? drow % pr.dl_T : 0;
        int half = 0;
#pragma unroll 1
        for (int c = 0; c < BLOCK_N; c += 64, half ^= 1) {
          if (n0 + c >= pr.N) break;                  // warp-uniform
          // staging: one buffer per chunk, or (GELU) a pair: pre-activation and activation tile of the same chunk
          uint8_t* buf = my_stage + sbuf * 4096;
          uint8_t* buf2 = buf + 4096;
          sbuf = (sbuf + (gelu ? 2 : 1)) % EPI_BUFS;
          if (lane == 0) { if (gelu) bulk_wait_read<EPI_BUFS / 2 - 1>(); else bulk_wait_read<EPI_BUFS - 1>(); }
          __syncwarp();
          uint8_t* rowp = buf + lane * 128;
          uint32_t r64[64];                            // both halves of the chunk in flight before one wait
          tmem_ld32_nowait(taddr + c, r64);
          tmem_ld32_nowait(taddr + c + 32, r64 + 32);
          uint4 ov[with_delta ? 8 : 1];               // this row's 64 values of O (head (n0 + c) / 64)
          if (with_delta) {
#pragma unroll
            for (int k = 0; k < 8; ++k)
              ov[k] = drow_ok ? __ldg(reinterpret_cast<const uint4*>(dl_orow + c) + k) : make_uint4(0, 0, 0, 0);
          }
          float dacc[4] = {0.f, 0.f, 0.f, 0.f};
          // the chunk's 64 bias values go to registers up front: interleaved with the (volatile, memory-
          // clobbering) st.shared they serialised into 8 load -> add -> store chains, 0.4 us per chunk
          float4 bq[16];
          const float* bsrc = my_bias + half * 64;
#pragma unroll
          for (int k = 0; k < 16; ++k) bq[k] = *reinterpret_cast<const float4*>(bsrc + 4 * k);
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
              if (with_delta) {                        // dO as stored (rounded to bf16) times O, fp32 accumulation
                const uint4 o4 = ov[4 * h + i];
                const uint32_t ow[4] = {o4.x, o4.y, o4.z, o4.w};
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                  dacc[u] = fmaf(__uint_as_float(w[u] << 16), __uint_as_float(ow[u] << 16), dacc[u]);
                  dacc[u] = fmaf(__uint_as_float(w[u] & 0xffff0000u), __uint_as_float(ow[u] & 0xffff0000u), dacc[u]);
                }
              }
              if (gelu) {                              // gelu of the ROUNDED pre-activation, as backward will see it
                uint32_t gw[4];
#pragma unroll
                for (int u = 0; u < 4; ++u)
                  gw[u] = pack_bf16x2(gelu_bf16(__uint_as_float(w[u] << 16)), gelu_bf16(__uint_as_float(w[u] & 0xffff0000u)));
                sts128(buf2 + lane * 128 + off, gw[0], gw[1], gw[2], gw[3]);
              }
            }
          }
          if (c + 64 < BLOCK_N) {                      // next chunk's bias -> the other half (c is warp-uniform)
            const int i2 = (c >> 5) + 2;
            float nb0 = 0.f, nb1 = 0.f;
#pragma unroll
            for (int i = 2; i < BLOCK_N / 32; i += 2)
              if (i == i2) { nb0 = breg[i]; nb1 = breg[i + 1]; }
            my_bias[(half ^ 1) * 64 + lane] = nb0;
            my_bias[(half ^ 1) * 64 + 32 + lane] = nb1;
          }
          if (with_delta && drow_ok) {
            const size_t idx = ((size_t)dl_b * pr.dl_H + ((n0 + c) >> 6)) * pr.dl_T + dl_t;
            pr.dl_delta[idx] = (dacc[0] + dacc[1]) + (dacc[2] + dacc[3]);
            pr.dl_lse2[idx] = __ldg(pr.dl_lse + idx) * LOG2E_F;
          }
          fence_async_smem();                         // generic-proxy writes -> visible to the TMA engine
          __syncwarp();
          if (lane == 0) {
            tma_store_2d(tmC, buf, n0 + c, m0 + q * 32);
            if (gelu) tma_store_2d(&maps.c2, buf2, n0 + c, m0 + q * 32);
            bulk_commit();
          }
        }
        };
        if (pr.gelu) chunks(std::integral_constant<int, 1>{});
        else if (pr.dl_o != nullptr) chunks(std::integral_constant<int, 2>{});
        else chunks(std::integral_constant<int, 0>{});
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(mapa_rank(smem_u32(&tempty[acc]), 0));
      acc ^= 1;
      if (acc == 0) acc_phase ^= 1;
    }
    if (lane == 0) bulk_wait_read<0>();               // smem must outlive the last TMA read; the global writes are
                                                      // complete at kernel end like any other store
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();                                  // no CTA leaves while its pair can still signal it
  if (warp == 5) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(TMEM_COLS) : "memory");
  }
  cluster_sync_all();                                  // pair-wide dealloc: neither CTA exits before both freed
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


template <int BLOCK_N, int STAGES>
int launch(const Maps& maps, const Params& p, int grid, cudaStream_t s) {
  constexpr size_t SMEM = (size_t)STAGES * (BLOCK_M * BLOCK_K * 2 + (BLOCK_N / 2) * BLOCK_K * 2) + EPI_STAGING_BYTES +
                          4 * 128 * 4 + 256;
  static_assert(SMEM <= 232448, "shared memory budget of one sm_100 CTA");
  auto kern = gemm_tc_kernel<BLOCK_N, STAGES>;
  { int rc_ = set_max_dynamic_smem((const void*)kern, (int)SMEM); if (rc_) return rc_; }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(NUM_THREADS);
  cfg.dynamicSmemBytes = SMEM;
  cfg.stream = s;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = 2;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[1].val.programmaticStreamSerializationAllowed = PACI_PDL_ATTR;
  cfg.attrs = attr;
  cfg.numAttrs = 2;
  PACI_CUDA_OK(cudaLaunchKernelEx(&cfg, kern, maps, p));
  g_launches.fetch_add(1, std::memory_order_relaxed);
  return PACI_OK;
}

thread_local int32_t g_last_plan[6] = {0, 0, 0, 0, 0, 0};

// validates one problem and fills its Prob + tensor maps
int fill_problem(const GemmDesc& d, int BN, Prob* pr, CUtensorMap* tmA, CUtensorMap* tmB, CUtensorMap* tmC,
                 CUtensorMap* tmC2) {
  if (d.gelu_out != nullptr && (d.out_f32_accum || (uintptr_t)d.gelu_out % 16))
    return fail(PACI_EINVAL, "tcgen05 GEMM: gelu output needs the bf16 epilogue and a 16-byte aligned pointer");
  if (d.K <= 0) return fail(PACI_EINVAL, "tcgen05 GEMM: K=%d", d.K);
  if (d.layout < 0 || d.layout > 2) return fail(PACI_EINVAL, "gemm: layout %d", d.layout);
  if ((uintptr_t)d.C % 16 || (d.out_f32_accum ? d.ldc % 4 : d.ldc % 8))
    return fail(PACI_EINVAL, "tcgen05 GEMM: C not 16-byte aligned (ldc=%d)", d.ldc);
  if (d.bias != nullptr && (uintptr_t)d.bias % 16) return fail(PACI_EINVAL, "tcgen05 GEMM: bias not 16-byte aligned");
  const bool a_mn = d.layout == 2, b_mn = d.layout != 0;
  int rc;
  // A: K-major [M rows][K contiguous] -> dims {K, M}, box {64, 128};  MN-major [K rows][M contiguous] -> {M, K}, {64, 64}
  rc = a_mn ? make_map(tmA, d.A, d.M, d.K, d.lda, 64, BLOCK_K) : make_map(tmA, d.A, d.K, d.M, d.lda, BLOCK_K, BLOCK_M);
  if (rc) return rc;
  rc = b_mn ? make_map(tmB, d.B, d.N, d.K, d.ldb, 64, BLOCK_K) : make_map(tmB, d.B, d.K, d.N, d.ldb, BLOCK_K, BN / 2);
  if (rc) return rc;
  // C: box of 32 rows x 128 bytes, written by one epilogue warp per TMA store / reduce-add
  rc = d.out_f32_accum ? make_map(tmC, d.C, d.N, d.M, d.ldc, 32, 32, 4) : make_map(tmC, d.C, d.N, d.M, d.ldc, 64, 32, 2);
  if (rc) return rc;
  if (d.gelu_out != nullptr && (rc = make_map(tmC2, d.gelu_out, d.N, d.M, d.ldc, 64, 32, 2))) return rc;
  pr->M = d.M; pr->N = d.N; pr->K = d.K;
  pr->tiles_m = ceil_div(d.M, BLOCK_M * 2);
  pr->tiles_n = ceil_div(d.N, BN);
  pr->kb_total = ceil_div(d.K, BLOCK_K);
  pr->splits = 1; pr->range_mode = 0;
  pr->a_mn = a_mn; pr->b_mn = b_mn; pr->accum = d.out_f32_accum != 0; pr->gelu = d.gelu_out != nullptr;
  pr->bias = d.bias;
  if (d.delta != nullptr) {
    const AttnDeltaOut& a = *d.delta;
    if (d.out_f32_accum || d.gelu_out != nullptr || d.N != a.H * 64 || a.T <= 0 || d.M % a.T != 0 || (uintptr_t)a.o % 16 ||
        a.ldo % 8 != 0)
      return fail(PACI_EINVAL, "tcgen05 GEMM: the delta epilogue needs the bf16 dgrad of an [mu T, H 64] output");
    pr->dl_o = a.o; pr->dl_ldo = a.ldo; pr->dl_lse = a.lse; pr->dl_delta = a.delta; pr->dl_lse2 = a.lse2;
    pr->dl_T = a.T; pr->dl_H = a.H;
  }
  return PACI_OK;
}

}  // namespace

int make_tensor_map(CUtensorMap* out, const void* ptr, uint64_t d0, uint64_t d1, uint64_t ld, uint32_t b0,
                    uint32_t b1, uint32_t esz) {
  return make_map(out, ptr, d0, d1, ld, b0, b1, esz);
}

// One launch for n <= 2 problems.  n == 2 is the backward pair of one linear layer: the wgrad (fp32 reduce-add output:
// arbitrarily divisible along its contraction) and the dgrad (bf16 output: whole tiles).  The dgrad's tiles are dealt
// round-robin over the CTA pairs, then the wgrad's (tile, k-block) units are poured on top until every pair carries
// the same number of k-blocks ("water-filling"), so the pair of GEMMs has ONE prologue, ONE pipeline fill, ONE exposed
// epilogue and no round quantisation (the 8192 x 1024 x 1024 dgrad alone: 128 tiles on 74 pairs = 1.73 rounds).
int gemm_tc_multi(const GemmDesc* d, int n, cudaStream_t s) {
  if (n < 1 || n > MAX_PROB) return fail(PACI_EINVAL, "gemm_tc_multi: n=%d", n);
  for (int i = 0; i < n; ++i)
    if (d[i].M <= 0 || d[i].N <= 0) {                  // an empty problem: launch the rest
      if (n == 1) return PACI_OK;
      return gemm_tc_multi(d + (i == 0 ? 1 : 0), 1, s);
    }
  if (n == 2) {
    const bool small0 = d[0].N <= 128, small1 = d[1].N <= 128;
    // the shared grid needs one tile width, the fp32 output first and no GELU output
    if (small0 != small1 || !d[0].out_f32_accum || d[1].out_f32_accum || d[0].gelu_out || d[1].gelu_out) {
      int rc = gemm_tc_multi(d, 1, s);
      return rc ? rc : gemm_tc_multi(d + 1, 1, s);
    }
  }
  const int BN = d[0].N <= 128 ? 128 : 256;
  Maps maps;
  Params p;
  std::memset(&p, 0, sizeof p);
  p.n_prob = n;
  for (int i = 0; i < n; ++i) {
    maps.c2 = maps.c[0];
    int rc = fill_problem(d[i], BN, &p.pr[i], &maps.a[i], &maps.b[i], &maps.c[i], &maps.c2);
    if (rc) return rc;
  }
  if (n == 1) { maps.a[1] = maps.a[0]; maps.b[1] = maps.b[0]; maps.c[1] = maps.c[0]; if (!d[0].gelu_out) maps.c2 = maps.c[0]; }
  const int workers = std::min(std::max(1, num_sms() / 2), MAX_WORKERS);
  int grid;
  if (n == 1) {
    Prob& pr = p.pr[0];
    const int tiles = pr.tiles_m * pr.tiles_n;
    int splits = 1;
    if (pr.accum) {
      // split-K over the contraction (tokens): partials meet in the fp32 TMA reduce-add epilogue.  Cost model in
      // k-block units: rounds of the persistent grid x (k-blocks per item + EPI), where EPI ~ 8 k-blocks stands
      // for an item's reduce-add epilogue (every extra split re-sends the whole fp32 tile through the L2 adders:
      // 8 splits of the 4096x1024 wgrad measured 73 us against 1 split's 1.73-round quantisation loss).
      const int max_s = std::max(1, std::min(pr.kb_total / 4, 32));
      const int EPI = 8;
      long best = -1;
      for (int sp = 1; sp <= max_s; ++sp) {
        const int kb_per = ceil_div(pr.kb_total, sp);
        if (ceil_div(pr.kb_total, kb_per) != sp) continue;        // every split owns at least one k-block
        const long rounds = ceil_div((long)tiles * sp, workers);
        const long cost = rounds * (kb_per + EPI);
        if (best < 0 || cost < best) { best = cost; splits = sp; }
      }
      // equal contiguous (tile, k-block) ranges instead of whole items: U / W k-blocks per worker plus one flush per
      // tile boundary crossed (+1).  Taken for outputs of many rounds (the LM-head wgrad: 788 tiles, 10.65 rounds ->
      // 0.659 to 0.597 ms); with fewer tiles than two rounds the k-block rate itself drops when every pair is busy
      // and the round-robin splits measured the same or better
      const long units = (long)tiles * pr.kb_total;
      const long per = ceil_div(units, (long)workers);
      const long cost = per + (ceil_div(per, (long)pr.kb_total) + 1) * EPI;
      const long item_cost = ceil_div((long)tiles * splits, (long)workers) * (ceil_div(pr.kb_total, splits) + EPI);
      if (tiles >= 2 * workers && cost < item_cost) {
        pr.range_mode = 1;
        for (int w = 0; w <= workers; ++w) p.ustart[0][w] = (int)(units * w / workers);
      }
    }
    pr.splits = splits;
    // balanced persistent grid: the same number of rounds on the fewest workers (128 tiles on 74 pairs take 2
    // rounds; so do 64 pairs, and the other 20 SMs stay free for the other stage streams' kernels)
    const int items = tiles * splits;
    const int rounds = ceil_div(items, workers);
    grid = (pr.range_mode ? workers : ceil_div(items, rounds)) * 2;
    g_last_plan[0] = 2; g_last_plan[1] = BN; g_last_plan[2] = splits; g_last_plan[3] = pr.range_mode;
    g_last_plan[4] = grid; g_last_plan[5] = tiles;
  } else {
    // problem 0 = wgrad (range mode, poured second), problem 1 = dgrad (whole tiles, round-robin).  The kernel walks
    // the wgrad range FIRST so that the launch's last, exposed epilogue is the cheaper bf16 store.
    Prob& wg = p.pr[0];
    Prob& dg = p.pr[1];
    const int tiles_d = dg.tiles_m * dg.tiles_n;
    const long U = (long)wg.tiles_m * wg.tiles_n * wg.kb_total;
    std::vector<long> load(workers);
    long total = U;
    for (int w = 0; w < workers; ++w) {
      load[w] = (long)((tiles_d - w + workers - 1) / workers) * dg.kb_total;   // tiles w, w + W, ...
      if (tiles_d <= w) load[w] = 0;
      total += load[w];
    }
    // water level T: sum_w max(0, T - load[w]) = U
    std::vector<long> sorted(load);
    std::sort(sorted.begin(), sorted.end());
    double level = 0.0;
    {
      long acc = 0;
      for (int i = 0; i < workers; ++i) {               // the i + 1 lightest workers fill up to `level`
        acc += sorted[i];
        level = (double)(U + acc) / (double)(i + 1);
        if (i + 1 == workers || level <= (double)sorted[i + 1]) break;
      }
    }
    double cum = 0.0;
    p.ustart[0][0] = 0;
    for (int w = 0; w < workers; ++w) {
      cum += std::max(0.0, level - (double)load[w]);
      p.ustart[0][w + 1] = (int)std::min<long>(U, (long)std::llround(cum));
    }
    p.ustart[0][workers] = (int)U;
    wg.range_mode = 1;
    dg.range_mode = 0; dg.splits = 1;
    grid = workers * 2;
    g_last_plan[0] = 2; g_last_plan[1] = BN; g_last_plan[2] = 2; g_last_plan[3] = 2;
    g_last_plan[4] = grid; g_last_plan[5] = tiles_d + wg.tiles_m * wg.tiles_n;
    (void)total;
  }
  if (BN == 128) return launch<128, 6>(maps, p, grid, s);
  return launch<256, 5>(maps, p, grid, s);
}

int gemm_tc(int layout, int M, int N, int K, const void* A, int lda, const void* B, int ldb, const float* bias,
            void* C, int ldc, int out_f32_accum, cudaStream_t s, void* gelu_out) {
  GemmDesc d{layout, M, N, K, A, lda, B, ldb, bias, C, ldc, out_f32_accum, gelu_out};
  return gemm_tc_multi(&d, 1, s);
}

void gemm_tc_last_plan(int32_t* out6) {
  for (int i = 0; i < 6; ++i) out6[i] = g_last_plan[i];
}

}  // namespace paci
