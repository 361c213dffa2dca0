// attention_tc.cu -- fused causal attention on the 5th-generation tensor cores (tcgen05 + TMEM + TMA),
// bf16, head dim 64, T a multiple of 128 (rows a4, a17 of SURVEY.md 8(a)).
//
// Forward.  One CTA = 128 query rows of one (batch, head); key blocks of 128; two CTAs per SM (115 KB of
// shared memory and 256 TMEM columns each), so one CTA's softmax overlaps the other CTA's MMAs.
//   warp 0     TMA producer: Q once, then K_j / V_j through 2-stage rings (one 2D tensor map over the packed
//              qkv tensor [mu*T, 3D], box 64 columns x 128 rows, 128-byte swizzle)
//   warp 1     MMA issuer (one thread): S = Q K_j^T (M128 N128 K64) into TMEM columns 0..127, then
//              O += P_j V_j (M128 N64 K128) into columns 128..191; S_{j+1} is issued before P_j V_j so the
//              tensor pipe always has the next scores ready
//   warps 2-5  softmax: thread = query row (TMEM lane).  One pass over S: tcgen05.ld 128 columns, row max,
//              p = exp2(s * c - m_ref), row sum, P as bf16 into 128B-swizzled shared memory (the A operand of
//              P V).  O stays in TMEM across key blocks (accumulate = 1) and is rescaled only when the running
//              max has grown by more than 2^8 since the reference max m_ref was taken ("lazy rescale"): the
//              final O / l and lse = m_ref + log2 l do not depend on which reference was used.
// qkv is packed [mu, T, 3D]: q | k | v, head h at columns h*64 .. h*64+63 (R17).
#include "tc_ptx.cuh"

namespace paci {

namespace {

using namespace tc;

constexpr int DH = 64;
constexpr float LOG2E = 1.4426950408889634f;
constexpr float LN2 = 0.6931471805599453f;

__device__ __forceinline__ void tmem_ld32_nowait(uint32_t taddr, uint32_t* r) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
        "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
        "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
        "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
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
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
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
constexpr uint32_t FWD_SMEM = TILE_BYTES * (1 + 2 + 2) + 2 * TILE_BYTES + 256;   // Q, K[2], V[2], P (2 tiles), barriers

__global__ void __launch_bounds__(FWD_THREADS, 2)
attn_fwd_tc_kernel(const __grid_constant__ CUtensorMap tm, int T, int H, bf16* __restrict__ o,
                   float* __restrict__ lse) {
  extern __shared__ __align__(1024) uint8_t smem[];
  uint8_t* sQ = smem;
  uint8_t* sK = sQ + TILE_BYTES;
  uint8_t* sV = sK + 2 * TILE_BYTES;
  uint8_t* sP = sV + 2 * TILE_BYTES;
  uint64_t* bars = (uint64_t*)(sP + 2 * TILE_BYTES);
  uint64_t *q_full = bars, *k_full = bars + 1, *v_full = bars + 3, *k_empty = bars + 5, *v_empty = bars + 7,
           *s_full = bars + 9, *p_full = bars + 10, *o_full = bars + 11;
  uint32_t* tmem_slot = (uint32_t*)(bars + 12);

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
    mbar_init(s_full, 1); mbar_init(p_full, 128); mbar_init(o_full, 1);
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
  const uint32_t tS = tmem_base, tO = tmem_base + 128;

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
      const uint32_t aQ = smem_u32(sQ), aP = smem_u32(sP);
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
        mbar_wait(p_full, (uint32_t)j & 1u, 15);           // P_j is in shared memory and S_j has been consumed
        tc_fence_after();
        if (j + 1 < n_kb) issue_qk(j + 1);
        const int st = j & 1;
        mbar_wait(&v_full[st], (uint32_t)(j >> 1) & 1u, 16);
        tc_fence_after();
        const uint32_t aV = smem_u32(sV + st * TILE_BYTES);
#pragma unroll
        for (int ks = 0; ks < 8; ++ks)                    // 8 x 16 keys
          umma_bf16(tO, smem_desc(aP + (ks >> 2) * TILE_BYTES + (ks & 3) * 32, 16, 1024),
                    smem_desc(aV + (ks >> 2) * 8192 + (ks & 3) * 2048, 8192, 1024), ID_PV, (j > 0 || ks > 0) ? 1u : 0u);
        umma_commit(&v_empty[st]);
        umma_commit(o_full);
      }
    }
  } else {
    const int r = (warp & 3) * 32 + lane;                 // query row inside the tile = TMEM lane
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
    const float c = rsqrtf((float)DH) * LOG2E;
    float m_ref = -INFINITY, l = 0.f;
    uint8_t* prow = sP + r * 128;
    for (int j = 0; j < n_kb; ++j) {
      mbar_wait(s_full, (uint32_t)j & 1u, 17);
      tc_fence_after();
      uint32_t s[128];
#pragma unroll
      for (int q = 0; q < 4; ++q) tmem_ld32_nowait(tS + lane_off + q * 32, s + q * 32);
      tmem_ld_wait();
      const bool diag = j == n_kb - 1;
      float mx = -INFINITY;
#pragma unroll
      for (int i = 0; i < 128; ++i) {
        float v = __uint_as_float(s[i]) * c;
        if (diag && i > r) v = -INFINITY;
        s[i] = __float_as_uint(v);
        mx = fmaxf(mx, v);
      }
      // lazy rescale (warp-uniform branch: tcgen05.ld / st are warp-collective)
      const bool grow = mx > m_ref + 8.f;
      if (j == 0) {
        m_ref = mx;
      } else if (__any_sync(0xffffffffu, grow)) {
        const float f = grow ? ex2(m_ref - mx) : 1.f;
        if (grow) { m_ref = mx; l *= f; }
        mbar_wait(o_full, (uint32_t)(j - 1) & 1u, 18);     // P_{j-1} V_{j-1} (and everything before) is in TMEM
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
      float sum = 0.f;
#pragma unroll
      for (int ch = 0; ch < 16; ++ch) {                   // 16 chunks of 8 keys = 16 bytes of bf16
        uint32_t w[4];
#pragma unroll
        for (int t = 0; t < 4; ++t) {
          const float p0 = ex2(__uint_as_float(s[ch * 8 + 2 * t]) - m_ref);
          const float p1 = ex2(__uint_as_float(s[ch * 8 + 2 * t + 1]) - m_ref);
          sum += p0 + p1;
          w[t] = pack_bf16x2(p0, p1);
        }
        sts128(prow + (ch >> 3) * TILE_BYTES + (((ch & 7) ^ (r & 7)) << 4), w[0], w[1], w[2], w[3]);
      }
      l += sum;
      fence_async_smem();                                 // P visible to the tensor core's async proxy
      tc_fence_before();
      mbar_arrive(p_full);
    }
    // epilogue: O / l -> bf16, lse
    mbar_wait(o_full, (uint32_t)(n_kb - 1) & 1u, 19);
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

}  // namespace

int attention_fwd_tc(int mu, int T, int H, const void* qkv, void* o, float* lse, cudaStream_t s) {
  const int D = H * DH;
  CUtensorMap tm;
  int rc = make_tensor_map(&tm, qkv, 3 * (uint64_t)D, (uint64_t)mu * T, 3 * (uint64_t)D, 64, 128, 2);
  if (rc) return rc;
  static bool attr_set = false;
  if (!attr_set) {
    PACI_CUDA_OK(cudaFuncSetAttribute(attn_fwd_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FWD_SMEM));
    attr_set = true;
  }
  const int grid = (T / 128) * H * mu;
  PACI_LAUNCH(attn_fwd_tc_kernel, grid, FWD_THREADS, FWD_SMEM, s, tm, T, H, (bf16*)o, lse);
  return PACI_OK;
}

}  // namespace paci
