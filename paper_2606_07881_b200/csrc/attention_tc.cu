// attention_tc.cu -- fused causal attention on the 5th-generation tensor cores (tcgen05 + TMEM + TMA),
// bf16, head dim 64, T a multiple of 128 (rows a4, a17 of SURVEY.md 8(a)).
//
// Forward.  One CTA = 128 query rows of one (batch, head); key blocks of 128; two CTAs per SM (82 KB of
// shared memory and 256 TMEM columns each), so one CTA's softmax overlaps the other CTA's MMAs.
//   warp 0     TMA producer: Q once, then K_j / V_j through 2-stage rings (one 2D tensor map over the packed
//              qkv tensor [mu*T, 3D], box 64 columns x 128 rows, 128-byte swizzle)
//   warp 1     MMA issuer (one thread): S = Q K_j^T (M128 N128 K64) into TMEM columns 0..127, then
//              O += P_j V_j (M128 N64 K128) into columns 128..191; S_{j+1} is issued before P_j V_j so the
//              tensor pipe always has the next scores ready
//   warps 2-5  softmax: thread = query row (TMEM lane).  One pass over S: tcgen05.ld 128 columns, row max,
//              p = exp2(s * c - m_ref), row sum, P as packed bf16 back into TMEM (tcgen05.st), the A operand of
//              P V (no shared-memory round trip).  O stays in TMEM across key blocks (accumulate = 1) and is rescaled only when the running
//              max has grown by more than 2^8 since the reference max m_ref was taken ("lazy rescale"): the
//              final O / l and lse = m_ref + log2 l do not depend on which reference was used.
// qkv is packed [mu, T, 3D]: q | k | v, head h at columns h*64 .. h*64+63 (R17).
#include <cstdlib>
#include <type_traits>

#include "tc_ptx.cuh"

namespace paci {

namespace {

using namespace tc;

constexpr int DH = 64;
constexpr float LOG2E = 1.4426950408889634f;
constexpr float LN2 = 0.6931471805599453f;

__device__ __forceinline__ void tmem_ld16_nowait(uint32_t taddr, uint32_t* r) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
        "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr));
}
template <int N> __device__ __forceinline__ void tmem_ld_cols_nowait(uint32_t taddr, uint32_t* r) {
  static_assert(N == 16 || N == 32 || N == 64, "column count");
  if constexpr (N == 16) tmem_ld16_nowait(taddr, r);
  else {
#pragma unroll
    for (int q = 0; q < N / 32; ++q) tmem_ld32_nowait(taddr + q * 32, r + q * 32);
  }
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t* r) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
      "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "
      "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};"
      ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),
        "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]),
        "r"(r[16]), "r"(r[17]), "r"(r[18]), "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]),
        "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31])
      : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t* r) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
      "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
      ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),
        "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
      : "memory");
}
// tcgen05.mma with the A operand in TENSOR MEMORY (K-major only): lane = row, one 32-bit column = two bf16 of K
__device__ __forceinline__ void umma_bf16_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t bdesc, uint32_t idesc_,
                                             uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
      ::"r"(tmem_d), "r"(tmem_a), "l"(bdesc), "r"(idesc_), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
// sm_100 packed fp32 pairs (FFMA2 / FADD2 / FMUL2: one issue slot for two elements), used by the BACKWARD kernels'
// elementwise phases: exp2 argument and dS = P (dP - delta) on pairs, 125.3 -> 122.4 us and 123.8 -> 121.2 mJ per call.
// (In the forward kernel, at 168 registers, the same change cost register-pair moves and spills: 55 -> 63 us.)
__device__ __forceinline__ uint64_t f2_pack(float lo, float hi) {
  uint64_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void f2_unpack(uint64_t v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ uint64_t f2_fma(uint64_t a, uint64_t b, uint64_t c) {
  uint64_t r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}
__device__ __forceinline__ uint64_t f2_sub(uint64_t a, uint64_t b) {
  uint64_t r;
  asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ uint64_t f2_mul(uint64_t a, uint64_t b) {
  uint64_t r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ float ex2(float x) {
  float r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

// instruction descriptor: D fp32, A/B bf16, majors, N>>3 at bit 17, M>>4 at bit 24
__host__ __device__ constexpr uint32_t idesc(int M, int N, bool a_mn, bool b_mn) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((a_mn ? 1u : 0u) << 15) | ((b_mn ? 1u : 0u) << 16) |
         ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

// ============================================================================== forward
constexpr int FWD_THREADS = 192;
constexpr uint32_t TILE_BYTES = 128 * 128;              // 128 rows x 64 bf16
constexpr uint32_t FWD_SMEM = TILE_BYTES * (1 + 2 + 2) + 256;   // Q, K[2], V[2], barriers (P lives in TMEM)

__global__ void __launch_bounds__(FWD_THREADS, 2)
attn_fwd_tc_kernel(const __grid_constant__ CUtensorMap tm, int T, int H, bf16* __restrict__ o,
                   float* __restrict__ lse) {
  extern __shared__ __align__(1024) uint8_t smem[];
  uint8_t* sQ = smem;
  uint8_t* sK = sQ + TILE_BYTES;
  uint8_t* sV = sK + 2 * TILE_BYTES;
  uint64_t* bars = (uint64_t*)(sV + 2 * TILE_BYTES);
  uint64_t *q_full = bars, *k_full = bars + 1, *v_full = bars + 3, *k_empty = bars + 5, *v_empty = bars + 7,
           *s_full = bars + 9, *p_full = bars + 10, *o_full = bars + 11, *s_free = bars + 12;
  uint32_t* tmem_slot = (uint32_t*)(bars + 13);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int D = H * DH;
  const int nq = T / 128;
  const int per_q = H * (int)(gridDim.x / (nq * H));     // H * mu
  const int qt = nq - 1 - (int)blockIdx.x / per_q;       // heaviest (last) query tiles first
  const int rem = (int)blockIdx.x % per_q;
  const int h = rem % H, b = rem / H;
  const int q0 = qt * 128;
  const int n_kb = qt + 1;                               // causal: key blocks 0 .. qt

  if ((smem_u32(smem) & 1023u) != 0) __trap();           // the 128-byte swizzle needs 1024-byte aligned tiles
  if (threadIdx.x == 0) {
    mbar_init(q_full, 1);
    for (int i = 0; i < 2; ++i) { mbar_init(&k_full[i], 1); mbar_init(&v_full[i], 1); mbar_init(&k_empty[i], 1); mbar_init(&v_empty[i], 1); }
    mbar_init(s_full, 1); mbar_init(p_full, 128); mbar_init(o_full, 1); mbar_init(s_free, 128);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(256) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  PACI_PDL_SYNC;
  const uint32_t tS = tmem_base, tO = tmem_base + 128, tP = tmem_base + 192;   // P: 128 keys as bf16 = 64 columns

  if (warp == 0) {
    if (lane == 0) {
      asm volatile("prefetch.tensormap [%0];" ::"l"(&tm) : "memory");
      const int row0 = b * T;
      mbar_expect_tx(q_full, TILE_BYTES);
      tma_load_2d(sQ, &tm, q_full, h * DH, row0 + q0);
      for (int j = 0; j < n_kb; ++j) {
        const int st = j & 1;
        const uint32_t ph = (uint32_t)(j >> 1) & 1u;
        mbar_wait(&k_empty[st], ph ^ 1, 11);
        mbar_expect_tx(&k_full[st], TILE_BYTES);
        tma_load_2d(sK + st * TILE_BYTES, &tm, &k_full[st], D + h * DH, row0 + j * 128);
        mbar_wait(&v_empty[st], ph ^ 1, 12);
        mbar_expect_tx(&v_full[st], TILE_BYTES);
        tma_load_2d(sV + st * TILE_BYTES, &tm, &v_full[st], 2 * D + h * DH, row0 + j * 128);
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {
      constexpr uint32_t ID_QK = idesc(128, 128, false, false), ID_PV = idesc(128, 64, false, true);
      const uint32_t aQ = smem_u32(sQ);
      auto issue_qk = [&](int j) {
        const int st = j & 1;
        mbar_wait(&k_full[st], (uint32_t)(j >> 1) & 1u, 13);
        tc_fence_after();
        const uint32_t aK = smem_u32(sK + st * TILE_BYTES);
#pragma unroll
        for (int kk = 0; kk < 4; ++kk)
          umma_bf16(tS, smem_desc(aQ + kk * 32, 16, 1024), smem_desc(aK + kk * 32, 16, 1024), ID_QK, kk > 0 ? 1u : 0u);
        umma_commit(&k_empty[st]);
        umma_commit(s_full);
      };
      mbar_wait(q_full, 0, 14);
      issue_qk(0);
      for (int j = 0; j < n_kb; ++j) {
        if (j + 1 < n_kb) {                                // S_j sits in the softmax threads' registers: the next
          mbar_wait(s_free, (uint32_t)j & 1u, 20);          // scores are computed WHILE they do exp2 / pack
          tc_fence_after();
          issue_qk(j + 1);
        }
        mbar_wait(p_full, (uint32_t)j & 1u, 15);           // P_j is in shared memory
        tc_fence_after();
        const int st = j & 1;
        mbar_wait(&v_full[st], (uint32_t)(j >> 1) & 1u, 16);
        tc_fence_after();
        const uint32_t aV = smem_u32(sV + st * TILE_BYTES);
#pragma unroll
        for (int ks = 0; ks < 8; ++ks)                    // 8 x 16 keys
          umma_bf16_ts(tO, tP + ks * 8, smem_desc(aV + (ks >> 2) * 8192 + (ks & 3) * 2048, 8192, 1024), ID_PV,
                       (j > 0 || ks > 0) ? 1u : 0u);                 // P from tensor memory: 8 columns per K = 16
        umma_commit(&v_empty[st]);
        umma_commit(o_full);
      }
    }
  } else {
    const int r = (warp & 3) * 32 + lane;                 // query row inside the tile = TMEM lane
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
    const float c = rsqrtf((float)DH) * LOG2E;
    float m_ref = -INFINITY, l = 0.f;
    for (int j = 0; j < n_kb; ++j) {
      mbar_wait_many(s_full, (uint32_t)j & 1u, 17);
      tc_fence_after();
      uint32_t s[128];
#pragma unroll
      for (int q = 0; q < 4; ++q) tmem_ld32_nowait(tS + lane_off + q * 32, s + q * 32);
      tmem_ld_wait();
      tc_fence_before();
      mbar_arrive(s_free);                                // S may be overwritten by Q K_{j+1}^T
      const bool diag = j == n_kb - 1;
      // row max of the RAW scores with four independent chains (one chain of 128 dependent FMNMX costs ~500
      // cycles); the scale c > 0 is applied to the max and folded into the exp2 argument as one FFMA
      float mx4[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
      if (diag) {
#pragma unroll
        for (int i = 0; i < 128; ++i) {
          if (i > r) s[i] = __float_as_uint(-INFINITY);
          mx4[i & 3] = fmaxf(mx4[i & 3], __uint_as_float(s[i]));
        }
      } else {
#pragma unroll
        for (int i = 0; i < 128; ++i) mx4[i & 3] = fmaxf(mx4[i & 3], __uint_as_float(s[i]));
      }
      const float mx = fmaxf(fmaxf(mx4[0], mx4[1]), fmaxf(mx4[2], mx4[3])) * c;
      // lazy rescale (warp-uniform branch: tcgen05.ld / st are warp-collective)
      const bool grow = mx > m_ref + 8.f;
      if (j == 0) {
        m_ref = mx;
      } else if (__any_sync(0xffffffffu, grow)) {
        const float f = grow ? ex2(m_ref - mx) : 1.f;
        if (grow) { m_ref = mx; l *= f; }
        mbar_wait_many(o_full, (uint32_t)(j - 1) & 1u, 18);     // P_{j-1} V_{j-1} (and everything before) is in TMEM
        tc_fence_after();
#pragma unroll
        for (int q = 0; q < 2; ++q) {
          uint32_t ov[32];
          tmem_ld32(tO + lane_off + q * 32, ov);
#pragma unroll
          for (int i = 0; i < 32; ++i) ov[i] = __float_as_uint(__uint_as_float(ov[i]) * f);
          tmem_st32(tO + lane_off + q * 32, ov);
        }
        tmem_st_wait();
      }
      // P is single-buffered: P_{j-1} V_{j-1} must have retired before P_j overwrites it (the next scores are
      // ready early now, so this is no longer implied by the MMA issue order)
      if (j > 0) { mbar_wait_many(o_full, (uint32_t)(j - 1) & 1u, 30); tc_fence_after(); }
      float sum4[4] = {0.f, 0.f, 0.f, 0.f};
      const float neg_m = -m_ref;
      // P goes registers -> TENSOR MEMORY (packed bf16, this thread's lane) and is the A operand of P V from there
#pragma unroll
      for (int half = 0; half < 2; ++half) {
        uint32_t w[32];
#pragma unroll
        for (int t = 0; t < 32; ++t) {
          const float p0 = ex2(fmaf(__uint_as_float(s[half * 64 + 2 * t]), c, neg_m));       // exp2(-inf) = 0: masked
          const float p1 = ex2(fmaf(__uint_as_float(s[half * 64 + 2 * t + 1]), c, neg_m));
          sum4[t & 3] += p0 + p1;
          w[t] = pack_bf16x2(p0, p1);
        }
        tmem_st32(tP + lane_off + half * 32, w);
      }
      l += (sum4[0] + sum4[1]) + (sum4[2] + sum4[3]);
      tmem_st_wait();
      tc_fence_before();
      mbar_arrive(p_full);
    }
    // epilogue: O / l -> bf16, lse
    mbar_wait_many(o_full, (uint32_t)(n_kb - 1) & 1u, 19);
    tc_fence_after();
    const float inv = 1.f / l;
    bf16* orow = o + ((size_t)b * T + q0 + r) * D + h * DH;
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      uint32_t ov[32];
      tmem_ld32(tO + lane_off + q * 32, ov);
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        uint4 w;
        w.x = pack_bf16x2(__uint_as_float(ov[8 * i]) * inv, __uint_as_float(ov[8 * i + 1]) * inv);
        w.y = pack_bf16x2(__uint_as_float(ov[8 * i + 2]) * inv, __uint_as_float(ov[8 * i + 3]) * inv);
        w.z = pack_bf16x2(__uint_as_float(ov[8 * i + 4]) * inv, __uint_as_float(ov[8 * i + 5]) * inv);
        w.w = pack_bf16x2(__uint_as_float(ov[8 * i + 6]) * inv, __uint_as_float(ov[8 * i + 7]) * inv);
        *reinterpret_cast<uint4*>(orow + q * 32 + i * 8) = w;
      }
    }
    lse[((size_t)b * H + h) * T + q0 + r] = (m_ref + log2f(l)) * LN2;
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(256) : "memory");
  }
}

// ============================================================================== backward
// Two launches of ONE kernel template (deterministic, no atomics), both with this skeleton: two STATIONARY
// 128-row tiles X0, X1 and a stream of 64-row tile pairs Y0, Y1 (2-stage TMA ring); per step
//     T0 = X0 Y0^T,  T1 = X1 Y1^T            (M128 N64 K64, into TMEM)
//     E0, E1 = elementwise(T0, T1)           (thread = TMEM lane = stationary row; bf16 back into TMEM)
//     ACC0 += E0 Y1,  ACC1 += E1 Y0          (M128 N64 K64, A operand from TMEM, accumulators in TMEM)
//   DKDV (one CTA per 128-key block): X = K_j, V_j; Y = Q_i, dO_i over the query steps at or below the
//        diagonal.  T0 = S^T, T1 = dP^T, E0 = P^T, E1 = dS^T; ACC0 = dV = P^T dO, ACC1 = dK = dS^T Q.
//        lse and delta are indexed by the streamed (query) index: 2 x 256 B per step ride the same ring.
//   DQ   (one CTA per 128-query tile): X = Q_i, dO_i; Y = K_j, V_j over the key steps at or left of the
//        diagonal.  T0 = S, T1 = dP, E1 = dS; ACC1 = dQ = dS K.  lse, delta are per-thread scalars.
// with P = exp2(S c - lse log2e), dS = P o (dP - delta) / sqrt(dh); the probabilities are recomputed from the
// stashed q, k and lse -- no parameter is involved, so this is not the checkpointed variant of P:282.
// T_{t+1} is issued before ACC_t, so the tensor pipe computes the next scores while the 128 elementwise
// threads work; two CTAs (98 KB smem, 256 TMEM columns each) share an SM.
constexpr int BWD_EW = 2;                               // elementwise warpgroups: each thread owns 64/EW columns
constexpr int BWD_THREADS = 64 + 128 * BWD_EW;
constexpr uint32_t HALF_BYTES = 64 * 128;               // 64 rows x 64 bf16
// ring depth of the streamed tiles (P^T / dS^T live in TMEM, so 4 stages fit in half an SM's shared memory)
__host__ __device__ constexpr int bwd_stages(bool dkdv) { return dkdv ? 4 : 4; }
__host__ __device__ constexpr uint32_t bwd_smem(bool dkdv) {
  return 2 * TILE_BYTES + bwd_stages(dkdv) * (2 * HALF_BYTES + 512) + 256;   // P^T / dS^T live in TMEM
}

__device__ __forceinline__ void bulk_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// PERSISTENT: the grid is two CTAs per SM; each CTA takes (tile, head, batch) items off a global counter (heaviest
// tiles first), so barrier setup, the TMEM allocation and the descriptor fetches are paid once per CTA, the
// stationary tiles of the next item load while the last step of the current one is being reduced, and the tail of
// the launch is balanced dynamically.  `g` counts streamed steps over the CTA's whole life: the ring and the
// per-step barriers are indexed by it; x_full / acc_full / acc_empty / x_empty complete once per item.
template <bool DKDV, int EW>
__global__ void __launch_bounds__(64 + 128 * EW, 2)
attn_bwd_tc_kernel(const __grid_constant__ CUtensorMap mX0, const __grid_constant__ CUtensorMap mX1,
                   const __grid_constant__ CUtensorMap mY0, const __grid_constant__ CUtensorMap mY1, int T, int H, int mu,
                   const float* __restrict__ lse, const float* __restrict__ delta, bf16* __restrict__ dqkv,
                   float* __restrict__ Gbias, int* __restrict__ work_counter) {
  extern __shared__ __align__(1024) uint8_t smem[];
  constexpr uint32_t YST = 2 * HALF_BYTES;               // one ring stage: Y0, Y1 (1024-byte aligned tiles)
  uint8_t* sX0 = smem;
  uint8_t* sX1 = sX0 + TILE_BYTES;
  uint8_t* sY = sX1 + TILE_BYTES;
  constexpr int NST = bwd_stages(DKDV);
  uint8_t* sStat = sY + NST * YST;                       // per stage: lse2[64], delta[64] of the streamed rows
  uint64_t* bars = (uint64_t*)(sStat + NST * 512);
  uint64_t *x_full = bars, *y_full = bars + 1, *y_empty = bars + 1 + NST, *t_full = bars + 1 + 2 * NST, *e_full = t_full + 1,
           *e_empty = t_full + 2, *acc_full = t_full + 3, *t_free = t_full + 4, *x_empty = t_full + 5, *acc_empty = t_full + 6,
           *item_full = t_full + 7 /* [2] */, *t1_full = t_full + 9, *t1_free = t_full + 10;
  // t_full / t_free: T0 (the score tile S) landed / is in registers; t1_full / t1_free: the same for T1 (dP)
  uint32_t* tmem_slot = (uint32_t*)(t_full + 11);
  volatile int* item_slot = (volatile int*)(tmem_slot + 1);   // [2]

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int D = H * DH;
  const int nt = T / 128;
  const int per = H * mu;
  const int n_items = nt * per;
  // item -> (first stationary row, head, first token row of the batch element, streamed range)
  struct Item { int x0, h, row0, c_begin, n_steps, bh; };
  auto decode = [&](int item) {
    Item it;
    const int rank = item / per, rem = item % per;       // heaviest tiles first
    const int tile = DKDV ? rank : nt - 1 - rank;
    it.h = rem % H;
    const int b = rem / H;
    it.x0 = tile * 128;                                  // first stationary row (key for DKDV, query for DQ)
    it.c_begin = DKDV ? it.x0 : 0;                       // streamed rows [c_begin, c_end), 64 per step
    it.n_steps = ((DKDV ? T : it.x0 + 128) - it.c_begin) / 64;
    it.row0 = b * T;
    it.bh = b * H + it.h;
    return it;
  };

  if ((smem_u32(smem) & 1023u) != 0) __trap();
  if (threadIdx.x == 0) {
    mbar_init(x_full, 1);
    for (int i = 0; i < NST; ++i) { mbar_init(&y_full[i], 1); mbar_init(&y_empty[i], 1); }
    mbar_init(t_full, 1); mbar_init(e_full, 128 * EW); mbar_init(e_empty, 1); mbar_init(acc_full, 1); mbar_init(t_free, 128 * EW);
    mbar_init(t1_full, 1); mbar_init(t1_free, 128 * EW);
    mbar_init(x_empty, 1); mbar_init(acc_empty, 128 * EW); mbar_init(&item_full[0], 1); mbar_init(&item_full[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(256) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  PACI_PDL_SYNC;
  const uint32_t tT0 = tmem_base, tT1 = tmem_base + 64, tA0 = tmem_base + 128, tA1 = tmem_base + 192;
  const uint32_t tE = tmem_base + 128;                   // DQ only (no dV accumulator there): dS as bf16, 32 columns

  if (warp == 0) {
    if (lane == 0) {
      uint32_t g = 0;
      for (uint32_t k = 0;; ++k) {
        // the slot of item k-2 is free: every consumer copied it before item k-1's stationary tiles could be
        // requested (x_empty of k-2), which happened before this point
        const int item = atomicAdd(work_counter, 1);
        item_slot[k & 1] = item;
        mbar_arrive(&item_full[k & 1]);                  // release: the slot write is visible to the waiters
        if (item >= n_items) break;
        const Item it = decode(item);
        // column of each operand inside its tensor: qkv = [q | k | v], dO = [D]
        const int cx0 = DKDV ? D + it.h * DH : it.h * DH;        // K_j | Q_i
        const int cx1 = DKDV ? 2 * D + it.h * DH : it.h * DH;    // V_j | dO_i
        const int cy0 = DKDV ? it.h * DH : D + it.h * DH;        // Q   | K
        const int cy1 = DKDV ? it.h * DH : 2 * D + it.h * DH;    // dO  | V
        mbar_wait(x_empty, (k & 1u) ^ 1u, 20);           // the previous item's score MMAs have read X
        mbar_expect_tx(x_full, 2 * TILE_BYTES);
        tma_load_2d(sX0, &mX0, x_full, cx0, it.row0 + it.x0);
        tma_load_2d(sX1, &mX1, x_full, cx1, it.row0 + it.x0);
        const float* lrow = lse + (size_t)it.bh * T;
        const float* drow = delta + (size_t)it.bh * T;
        for (int t = 0; t < it.n_steps; ++t, ++g) {
          const int st = g % NST, c0 = it.c_begin + t * 64;
          mbar_wait(&y_empty[st], ((g / NST) & 1u) ^ 1u, 21);
          uint8_t* y = sY + st * YST;
          mbar_expect_tx(&y_full[st], 2 * HALF_BYTES + (DKDV ? 512u : 0u));
          tma_load_2d(y, &mY0, &y_full[st], cy0, it.row0 + c0);
          tma_load_2d(y + HALF_BYTES, &mY1, &y_full[st], cy1, it.row0 + c0);
          if (DKDV) {
            bulk_load_1d(sStat + st * 512, lrow + c0, 256, &y_full[st]);
            bulk_load_1d(sStat + st * 512 + 256, drow + c0, 256, &y_full[st]);
          }
        }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {
      constexpr uint32_t ID_T = idesc(128, 64, false, false), ID_ACC = idesc(128, 64, false, true);
      const uint32_t aX0 = smem_u32(sX0), aX1 = smem_u32(sX1);
      auto issue_t0 = [&](uint32_t gs) {
        const int st = gs % NST;
        mbar_wait(&y_full[st], (gs / NST) & 1u, 22);
        tc_fence_after();
        const uint32_t aY0 = smem_u32(sY + st * YST);
#pragma unroll
        for (int kk = 0; kk < 4; ++kk)
          umma_bf16(tT0, smem_desc(aX0 + kk * 32, 16, 1024), smem_desc(aY0 + kk * 32, 16, 1024), ID_T, kk > 0 ? 1u : 0u);
        umma_commit(t_full);
      };
      auto issue_t1 = [&](uint32_t gs) {                  // after issue_t0(gs): the stage is known to have landed
        const uint32_t aY1 = smem_u32(sY + (gs % NST) * YST) + HALF_BYTES;
#pragma unroll
        for (int kk = 0; kk < 4; ++kk)
          umma_bf16(tT1, smem_desc(aX1 + kk * 32, 16, 1024), smem_desc(aY1 + kk * 32, 16, 1024), ID_T, kk > 0 ? 1u : 0u);
        umma_commit(t1_full);
      };
      uint32_t g = 0;
      for (uint32_t k = 0;; ++k) {
        mbar_wait(&item_full[k & 1], (k >> 1) & 1u, 19);
        const int item = item_slot[k & 1];
        if (item >= n_items) break;
        const int n_steps = decode(item).n_steps;
        mbar_wait(x_full, k & 1u, 23);
        if (g > 0) {                                      // the previous item's last T0 / T1 are in registers
          mbar_wait(t_free, (g - 1) & 1u, 29);
          if (!DKDV) mbar_wait(t1_free, (g - 1) & 1u, 30);   // (dK/dV: implied by e_full, T1 goes behind the accumulates)
          tc_fence_after();
        }
        issue_t0(g);
        issue_t1(g);                                      // (dK/dV) in order behind the previous item's last accumulate MMAs
        if (k > 0) {                                      // the previous item's accumulators have been read out
          mbar_wait(acc_empty, (k - 1) & 1u, 18);
          tc_fence_after();
        }
        for (int t = 0; t < n_steps; ++t, ++g) {
          const bool more = t + 1 < n_steps;
          if (more) {                                     // T_t sits in the elementwise threads' registers: the next
            mbar_wait(t_free, g & 1u, 29);                // score-type MMAs run WHILE they do exp2 / pack
            tc_fence_after();
            issue_t0(g + 1);
            if (!DKDV) {
              mbar_wait(t1_free, g & 1u, 30);
              tc_fence_after();
              issue_t1(g + 1);
              if (t + 2 == n_steps) umma_commit(x_empty); // X is not read again: the next item's may load
            }
          }
          mbar_wait(e_full, g & 1u, 24);                  // E_t is in tensor memory
          tc_fence_after();
          const int st = g % NST;
          const uint32_t aY0 = smem_u32(sY + st * YST), aY1 = aY0 + HALF_BYTES;
          const uint32_t acc = t > 0 ? 1u : 0u;
          if (DKDV) {
            // P^T and dS^T (bf16) sit in T1's 64 columns: warpgroup g wrote its 32 queries of P^T at +32 g and of dS^T
            // at +32 g + 16; one K = 16 step of the A operand is 8 columns
#pragma unroll
            for (int kk = 0; kk < 4; ++kk)                // dV += P^T dO
              umma_bf16_ts(tA0, tT1 + 32 * (kk >> 1) + 8 * (kk & 1), smem_desc(aY1 + kk * 2048, 8192, 1024), ID_ACC, (acc | (kk > 0)) ? 1u : 0u);
#pragma unroll
            for (int kk = 0; kk < 4; ++kk)                // dK += dS^T Q
              umma_bf16_ts(tA1, tT1 + 32 * (kk >> 1) + 16 + 8 * (kk & 1), smem_desc(aY0 + kk * 2048, 8192, 1024), ID_ACC, (acc | (kk > 0)) ? 1u : 0u);
          } else {
#pragma unroll
            for (int kk = 0; kk < 4; ++kk)                // dQ += dS K, dS from its own TMEM columns
              umma_bf16_ts(tA1, tE + kk * 8, smem_desc(aY0 + kk * 2048, 8192, 1024), ID_ACC, (acc | (kk > 0)) ? 1u : 0u);
          }
          umma_commit(&y_empty[st]);
          umma_commit(e_empty);
          // dK/dV: T1_{t+1} overwrites the columns P^T / dS^T were read from, so it is issued AFTER the accumulate
          // MMAs of step t (the tensor pipe executes one thread's MMAs in order)
          if (DKDV && more) {
            issue_t1(g + 1);
            if (t + 2 == n_steps) umma_commit(x_empty);
          }
        }
        umma_commit(acc_full);
      }
    }
  } else {
    // EW warpgroups of 4 warps: warp w owns TMEM lanes 32 (w % 4) .., warpgroup g = (w - 2) / 4 owns columns
    // [g CW, (g + 1) CW) of T0 / T1 -- the backward has no row reductions, so the groups never talk.
    // `lse` here is lse * log2(e) (written by the delta kernel); the 1/sqrt(dh) of dS is applied once, to
    // the dK / dQ accumulators in the epilogue (exact: a power of two).
    constexpr int CW = 64 / EW;
    const int r = (warp & 3) * 32 + lane;                 // stationary row inside the tile = TMEM lane
    const int wg = (warp - 2) >> 2;
    const int cw0 = wg * CW;
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
    const float c = rsqrtf((float)DH) * LOG2E;
    const float inv_sqrt = rsqrtf((float)DH);
    // Gbias (fp32 [3D], may be NULL): the bias gradient of the QKV projection = column sums of dqkv over all
    // tokens (row a15), taken here from the ROUNDED values being stored: one warp-shuffle reduction over the
    // warp's 32 rows per column, then one atomic per column per warp -- no separate pass over dqkv.
    auto store_chunk = [&](uint32_t taddr, bf16* dst, float scale, float* gcol) {   // 32 fp32 columns -> 32 bf16
      uint32_t ov[32];
      tmem_ld32(taddr + lane_off, ov);
      float cs[32];                                       // the rounded values, for the column sums
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        uint4 w;
        w.x = pack_bf16x2(__uint_as_float(ov[8 * i]) * scale, __uint_as_float(ov[8 * i + 1]) * scale);
        w.y = pack_bf16x2(__uint_as_float(ov[8 * i + 2]) * scale, __uint_as_float(ov[8 * i + 3]) * scale);
        w.z = pack_bf16x2(__uint_as_float(ov[8 * i + 4]) * scale, __uint_as_float(ov[8 * i + 5]) * scale);
        w.w = pack_bf16x2(__uint_as_float(ov[8 * i + 6]) * scale, __uint_as_float(ov[8 * i + 7]) * scale);
        *reinterpret_cast<uint4*>(dst + i * 8) = w;
        const uint32_t ww[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          cs[8 * i + 2 * u] = __uint_as_float(ww[u] << 16);
          cs[8 * i + 2 * u + 1] = __uint_as_float(ww[u] & 0xffff0000u);
        }
      }
      if (gcol != nullptr) {
        // transposing butterfly: after the step with offset `off` a lane keeps the half of its columns selected by
        // that bit of its lane id, summed with its partner's; 16 + 8 + 4 + 2 + 1 shuffles leave lane l with the sum
        // of column l over the warp's 32 rows -> one coalesced atomic per warp
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) {
          const bool up = (lane & off) != 0;
#pragma unroll
          for (int i = 0; i < off; ++i) {
            const float keep = up ? cs[i + off] : cs[i];
            const float send = up ? cs[i] : cs[i + off];
            cs[i] = keep + __shfl_xor_sync(0xffffffffu, send, off);
          }
        }
        atomicAdd(gcol + lane, cs[0]);
      }
    };
    uint32_t g = 0;
#ifdef PACI_ATTN_TIMING
    long long tk[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0}, tprev = clock64(), tnow;
#define TICK(i) do { tnow = clock64(); tk[i] += tnow - tprev; tprev = tnow; } while (0)
#else
#define TICK(i) do {} while (0)
#endif
    for (uint32_t k = 0;; ++k) {
      mbar_wait_many(&item_full[k & 1], (k >> 1) & 1u, 17);
      TICK((k == 0 ? 8 : 5));
      const int item = item_slot[k & 1];
      if (item >= n_items) break;
      const Item it = decode(item);
      const int x0 = it.x0;
      float my_lse2 = 0.f, my_delta = 0.f;
      if (!DKDV) {
        my_lse2 = lse[(size_t)it.bh * T + x0 + r];
        my_delta = delta[(size_t)it.bh * T + x0 + r];
      }
      for (int t = 0; t < it.n_steps; ++t, ++g) {
        const int st = g % NST, c0 = it.c_begin + t * 64;
        // phase 1 needs only the scores: P = exp2(S c - lse2), masked on the diagonal steps.  It runs while the tensor
        // pipe is still busy with the previous step's accumulate MMAs and this step's T1 (which, for dK/dV, can only
        // be issued behind them).
        mbar_wait_many(t_full, g & 1u, 25);
        tc_fence_after();
        TICK((t == 0 ? (k == 0 ? 8 : 9) : 0));
        uint32_t s[CW];                                   // S, then P (fp32 bits)
        tmem_ld_cols_nowait<CW>(tT0 + lane_off + cw0, s);
        tmem_ld_wait();
        tc_fence_before();
        mbar_arrive(t_free);                              // T0 may be overwritten by the next step's score MMA
        const float4* pl = reinterpret_cast<const float4*>(sStat + st * 512) + cw0 / 4;   // lse2 of the step's 64 queries
        const float4* pd = pl + 16;                                                        // delta
        if (DKDV) mbar_wait_many(&y_full[st], (g / NST) & 1u, 26);   // the step's lse / delta have landed
        // causal keep: query >= key.  DKDV: query = c0 + col, key = x0 + r.  DQ: query = x0 + r, key = c0 + col.
        // Only the two diagonal steps need the mask; `rel` is the diagonal's column inside this thread's slice.
        const bool diag = DKDV ? (c0 < x0 + 128) : (c0 + 63 > x0);
        const int rel = x0 + r - c0 - cw0;
        uint32_t wp[CW / 2], wd[CW / 2];
        auto phase1 = [&](auto masked) {
#pragma unroll
          for (int k4 = 0; k4 < CW / 4; ++k4) {
            float l2[4] = {my_lse2, my_lse2, my_lse2, my_lse2};
            if (DKDV) {
              const float4 a4 = pl[k4];
              l2[0] = a4.x; l2[1] = a4.y; l2[2] = a4.z; l2[3] = a4.w;
            }
#pragma unroll
            for (int e = 0; e < 4; e += 2) {
              const int i = 4 * k4 + e;
              float a0, a1;
              f2_unpack(f2_fma(f2_pack(__uint_as_float(s[i]), __uint_as_float(s[i + 1])), f2_pack(c, c),
                               f2_pack(-l2[e], -l2[e + 1])), a0, a1);
              float pr0 = ex2(a0), pr1 = ex2(a1);
              if (decltype(masked)::value) {
                const bool keep0 = DKDV ? (i >= rel) : (i <= rel);
                const bool keep1 = DKDV ? (i + 1 >= rel) : (i + 1 <= rel);
                pr0 = keep0 ? pr0 : 0.f;
                pr1 = keep1 ? pr1 : 0.f;
              }
              s[i] = __float_as_uint(pr0);
              s[i + 1] = __float_as_uint(pr1);
            }
            if (DKDV) {
              wp[2 * k4] = pack_bf16x2(__uint_as_float(s[4 * k4]), __uint_as_float(s[4 * k4 + 1]));
              wp[2 * k4 + 1] = pack_bf16x2(__uint_as_float(s[4 * k4 + 2]), __uint_as_float(s[4 * k4 + 3]));
            }
          }
        };
        if (diag) phase1(std::true_type{}); else phase1(std::false_type{});
        TICK(1);
        // phase 2: dS = P o (dP - delta), in two halves to keep the register footprint down
        mbar_wait_many(t1_full, g & 1u, 31);
        tc_fence_after();
        TICK(2);
#pragma unroll
        for (int hf = 0; hf < 2; ++hf) {
          uint32_t dp[CW / 2];
          tmem_ld_cols_nowait<CW / 2>(tT1 + lane_off + cw0 + hf * (CW / 2), dp);
          tmem_ld_wait();
#pragma unroll
          for (int k4 = 0; k4 < CW / 8; ++k4) {
            float dl[4] = {my_delta, my_delta, my_delta, my_delta};
            if (DKDV) {
              const float4 d4 = pd[hf * (CW / 8) + k4];
              dl[0] = d4.x; dl[1] = d4.y; dl[2] = d4.z; dl[3] = d4.w;
            }
            float dv[4];
#pragma unroll
            for (int e = 0; e < 4; e += 2) {
              const int i = 4 * k4 + e;
              f2_unpack(f2_mul(f2_pack(__uint_as_float(s[hf * (CW / 2) + i]), __uint_as_float(s[hf * (CW / 2) + i + 1])),
                               f2_sub(f2_pack(__uint_as_float(dp[i]), __uint_as_float(dp[i + 1])), f2_pack(dl[e], dl[e + 1]))),
                        dv[e], dv[e + 1]);
            }
            wd[hf * (CW / 4) + 2 * k4] = pack_bf16x2(dv[0], dv[1]);
            wd[hf * (CW / 4) + 2 * k4 + 1] = pack_bf16x2(dv[2], dv[3]);
          }
        }
        if (!DKDV) {                                      // (dK/dV: e_full says as much)
          tc_fence_before();
          mbar_arrive(t1_free);                           // T1 may be overwritten by the next step's dP MMA
        }
        if (g > 0) mbar_wait_many(e_empty, (g - 1) & 1u, 27);                  // the previous accumulate MMAs have read E
        TICK(3);
        // P^T / dS^T go to TENSOR MEMORY (the thread's lane, CW/2 packed columns each) and are the A operands of the
        // accumulate MMAs straight from there: no shared-memory round trip, no proxy fence.  dK/dV: they overwrite
        // this thread's own 32 columns of T1 (already in its registers); dQ: dS has columns of its own.
        static_assert(CW == 32, "tcgen05.st x16 per thread");
        if (DKDV) {
          tmem_st16(tT1 + lane_off + cw0, wp);
          tmem_st16(tT1 + lane_off + cw0 + 16, wd);
        } else {
          tmem_st16(tE + lane_off + cw0 / 2, wd);
        }
        tmem_st_wait();
        tc_fence_before();
        mbar_arrive(e_full);
        TICK(4);
      }
      // epilogue: accumulators -> bf16 rows of dqkv, 32-column chunks dealt round-robin to the warpgroups
      mbar_wait_many(acc_full, k & 1u, 28);
      tc_fence_after();
      TICK(6);
      bf16* orow = dqkv + ((size_t)it.row0 + x0 + r) * 3 * D + it.h * DH;
      constexpr int N_CHUNKS = DKDV ? 4 : 2;              // DKDV: dV lo, dV hi, dK lo, dK hi.  DQ: dQ lo, dQ hi
      for (int q = wg; q < N_CHUNKS; q += EW) {           // warp-uniform
        if (DKDV) {
          const int col = (q < 2 ? 2 * D : D) + (q & 1) * 32;
          store_chunk((q < 2 ? tA0 : tA1) + (q & 1) * 32, orow + col, q < 2 ? 1.f : inv_sqrt,
                      Gbias != nullptr ? Gbias + it.h * DH + col : nullptr);
        } else {
          store_chunk(tA1 + q * 32, orow + q * 32, inv_sqrt, Gbias != nullptr ? Gbias + it.h * DH + q * 32 : nullptr);
        }
      }
      tc_fence_before();
      mbar_arrive(acc_empty);                             // the next item's first accumulate MMA may overwrite them
      TICK(7);
    }
#ifdef PACI_ATTN_TIMING
    if (threadIdx.x == 64 && (blockIdx.x == 0 || blockIdx.x == 150 || blockIdx.x == 295))
      printf("bwd dkdv=%d blk %d steps %u items: per step: wait_t0 %lld phase1 %lld wait_t1 %lld phase2+wait_e %lld st+arrive %lld | total: prologue %lld item_wait %lld first_t0 %lld acc_wait %lld epilogue %lld\n",
             (int)DKDV, (int)blockIdx.x, g, tk[0] / g, tk[1] / g, tk[2] / g, tk[3] / g, tk[4] / g, tk[8], tk[5], tk[9], tk[6], tk[7]);
#endif
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(256) : "memory");
  }
}


// delta[b,h,t] = sum_d dO[b,t,h,d] * O[b,t,h,d]: 8 threads per (b,t,h), one 16-byte vector each
__global__ void __launch_bounds__(256) attn_delta_tc_kernel(size_t n_vec, int T, int H, const bf16* __restrict__ dout,
                                                            const bf16* __restrict__ o, const float* __restrict__ lse,
                                                            float* __restrict__ delta, float* __restrict__ lse2,
                                                            int* __restrict__ work_counters) {
  PACI_PDL_SYNC;
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < 2) work_counters[i] = 0;                        // item counters of the two persistent backward kernels
  float acc = 0.f;
  if (i < n_vec) {
    float a[8], c[8];
    load_vec<bf16>(dout + i * 8, a);
    load_vec<bf16>(o + i * 8, c);
#pragma unroll
    for (int j = 0; j < 8; ++j) acc += a[j] * c[j];
  }
#pragma unroll
  for (int sh = 1; sh < 8; sh <<= 1) acc += __shfl_xor_sync(0xffffffffu, acc, sh);
  if (i < n_vec && (threadIdx.x & 7) == 0) {
    const size_t hv = i >> 3;                  // (b*T + t)*H + h
    const size_t bt = hv / H;
    const size_t idx = ((bt / T) * H + hv % H) * T + bt % T;
    delta[idx] = acc;
    lse2[idx] = lse[idx] * LOG2E;                         // the backward kernels work in the exp2 domain
  }
}

}  // namespace

// delta, lse2 (fp32 [mu, H, T] each) and the two work counters of the persistent kernels
size_t attention_bwd_tc_scratch_bytes(int mu, int T, int H) { return 2 * (size_t)mu * H * T * sizeof(float) + 64; }

// scratch_prepared: delta and lse2 are already in `scratch` (written by the out-projection dgrad's epilogue,
// AttnDeltaOut); only the two work counters are reset here.
int attention_bwd_tc(int mu, int T, int H, const void* dout, const void* qkv, const void* o, const float* lse,
                     void* dqkv, float* scratch, float* Gbias, int scratch_prepared, cudaStream_t s) {
  const int D = H * DH;
  const uint64_t rows = (uint64_t)mu * T;
  CUtensorMap q128, q64, d128, d64;
  int rc;
  if ((rc = make_tensor_map(&q128, qkv, 3 * (uint64_t)D, rows, 3 * (uint64_t)D, 64, 128, 2))) return rc;
  if ((rc = make_tensor_map(&q64, qkv, 3 * (uint64_t)D, rows, 3 * (uint64_t)D, 64, 64, 2))) return rc;
  if ((rc = make_tensor_map(&d128, dout, (uint64_t)D, rows, (uint64_t)D, 64, 128, 2))) return rc;
  if ((rc = make_tensor_map(&d64, dout, (uint64_t)D, rows, (uint64_t)D, 64, 64, 2))) return rc;
  { int rc_ = set_max_dynamic_smem((const void*)attn_bwd_tc_kernel<true, BWD_EW>, (int)bwd_smem(true)); if (rc_) return rc_; }
  { int rc_ = set_max_dynamic_smem((const void*)attn_bwd_tc_kernel<false, BWD_EW>, (int)bwd_smem(false)); if (rc_) return rc_; }
  float* delta = scratch;
  float* lse2 = scratch + (size_t)mu * H * T;
  int* counters = reinterpret_cast<int*>(scratch + 2 * (size_t)mu * H * T);
  const size_t n_vec = (size_t)mu * T * D / 8;
  if (scratch_prepared) {
    PACI_CUDA_OK(cudaMemsetAsync(counters, 0, 2 * sizeof(int), s));
  } else {
    PACI_LAUNCH(attn_delta_tc_kernel, ceil_div((long long)n_vec, 256), 256, 0, s, n_vec, T, H, (const bf16*)dout,
                (const bf16*)o, lse, delta, lse2, counters);
  }
  const int n_sm = num_sms();
  const int items = (T / 128) * H * mu;
  const int grid = items < 2 * n_sm ? items : 2 * n_sm;   // persistent: two CTAs per SM
  // dK, dV: stationary K_j, V_j (qkv, 128-row boxes); streamed Q_i (qkv), dO_i (dout), 64-row boxes
  PACI_LAUNCH((attn_bwd_tc_kernel<true, BWD_EW>), grid, BWD_THREADS, bwd_smem(true), s, q128, q128, q64, d64, T, H, mu, lse2, delta,
              (bf16*)dqkv, Gbias, counters);
  // dQ: stationary Q_i (qkv), dO_i (dout); streamed K_j, V_j (qkv)
  PACI_LAUNCH((attn_bwd_tc_kernel<false, BWD_EW>), grid, BWD_THREADS, bwd_smem(false), s, q128, d128, q64, q64, T, H, mu, lse2, delta,
              (bf16*)dqkv, Gbias, counters + 1);
  return PACI_OK;
}

int attention_fwd_tc(int mu, int T, int H, const void* qkv, void* o, float* lse, cudaStream_t s) {
  const int D = H * DH;
  CUtensorMap tm;
  int rc = make_tensor_map(&tm, qkv, 3 * (uint64_t)D, (uint64_t)mu * T, 3 * (uint64_t)D, 64, 128, 2);
  if (rc) return rc;
  { int rc_ = set_max_dynamic_smem((const void*)attn_fwd_tc_kernel, (int)FWD_SMEM); if (rc_) return rc_; }
  const int grid = (T / 128) * H * mu;
  PACI_LAUNCH(attn_fwd_tc_kernel, grid, FWD_THREADS, FWD_SMEM, s, tm, T, H, (bf16*)o, lse);
  return PACI_OK;
}

}  // namespace paci
