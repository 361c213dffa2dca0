// attention_mma.cu -- fused causal attention forward / backward for bf16, head dim 64 (rows a4, a17).
//
// Flash-style: the T x T score matrix never leaves the SM.  Tiles of q/k/v are staged in shared
// memory by cp.async with a 128-byte XOR swizzle (conflict-free ldmatrix), the two contractions of
// every step run on the tensor cores (mma.sync.m16n8k16 bf16 -> fp32), the softmax statistics stay in
// fp32 registers (exp2 with the 1/sqrt(dh)*log2(e) scale folded in).  Backward recomputes the
// probabilities from the stashed q, k and lse -- no parameter is involved, so this is not the
// checkpointed variant of P:282 -- and is split into two deterministic kernels (no atomics):
//   dkdv: one CTA per 64-key block, loops over the query blocks at or below the diagonal
//   dq  : one CTA per 64-query block, loops over the key blocks at or left of the diagonal
// This version uses the legacy warp-level tensor-core path; a tcgen05/TMEM rewrite is the next step
// for this kernel.
//
// qkv is packed [mu, T, 3D]: q | k | v, head h at columns h*64 .. h*64+63 (R17).
#include "common.cuh"

namespace paci {

namespace {

constexpr int DH = 64;
constexpr float LOG2E = 1.4426950408889634f;
constexpr float LN2 = 0.6931471805599453f;

__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// 64-column bf16 tile, 128 bytes per row, 16-byte chunk c of row r stored at chunk (c ^ (r & 7))
__device__ __forceinline__ uint32_t tile_off(int row, int chunk) { return row * 128 + (((chunk ^ row) & 7) << 4); }

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

// rows x 64 bf16 tile from global (row stride ld elements) into swizzled smem, NT threads cooperate
template <int ROWS, int NT>
__device__ __forceinline__ void load_tile(uint32_t sbase, const bf16* g, size_t ld, int tid) {
#pragma unroll
  for (int i = tid; i < ROWS * 8; i += NT) {
    const int r = i >> 3, c = i & 7;
    cp_async16(sbase + tile_off(r, c), g + (size_t)r * ld + c * 8);
  }
}

__device__ __forceinline__ void ldsm_x4(uint32_t (&r)[4], uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t (&r)[4], uint32_t addr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void mma16816(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, "
      "{%0, %1, %2, %3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}

// A fragments (16 rows x 64 k) of a row-major tile: rows r0..r0+15 -> a[4 k-steps][4]
__device__ __forceinline__ void load_a_frags(uint32_t (&a)[4][4], uint32_t sbase, int r0, int lane) {
#pragma unroll
  for (int ks = 0; ks < 4; ++ks) ldsm_x4(a[ks], sbase + tile_off(r0 + (lane & 15), ks * 2 + (lane >> 4)));
}

// acc[8 n-tiles][4] (16 x 64, fp32) = A(16 x 64k) * B^T where B is a row-major [64 n][64 k] tile (n = rows)
__device__ __forceinline__ void mma_a_bT(float (&acc)[8][4], const uint32_t (&a)[4][4], uint32_t sB, int lane) {
#pragma unroll
  for (int ks = 0; ks < 4; ++ks) {
#pragma unroll
    for (int np = 0; np < 4; ++np) {   // pairs of n-tiles
      uint32_t b[4];
      ldsm_x4(b, sB + tile_off(np * 16 + (lane & 7) + ((lane >> 4) << 3), ks * 2 + ((lane >> 3) & 1)));
      mma16816(acc[2 * np], a[ks], b[0], b[1]);
      mma16816(acc[2 * np + 1], a[ks], b[2], b[3]);
    }
  }
}

// acc[8 n-tiles][4] (16 x 64) += P(16 x 64k, bf16 fragments in registers) * B where B is a row-major
// [64 k][64 n] tile (k = rows): fragments via ldmatrix.trans
__device__ __forceinline__ void mma_p_b(float (&acc)[8][4], const uint32_t (&p)[4][4], uint32_t sB, int lane) {
#pragma unroll
  for (int ks = 0; ks < 4; ++ks) {
#pragma unroll
    for (int np = 0; np < 4; ++np) {
      uint32_t b[4];
      ldsm_x4_t(b, sB + tile_off(ks * 16 + (lane & 7) + (((lane >> 3) & 1) << 3), np * 2 + (lane >> 4)));
      mma16816(acc[2 * np], p[ks], b[0], b[1]);
      mma16816(acc[2 * np + 1], p[ks], b[2], b[3]);
    }
  }
}

// accumulator layout (m16n8 tiles) -> A-operand fragments (m16k16), bf16
__device__ __forceinline__ void acc_to_a(uint32_t (&p)[4][4], const float (&s)[8][4]) {
#pragma unroll
  for (int ks = 0; ks < 4; ++ks) {
    p[ks][0] = pack_bf16(s[2 * ks][0], s[2 * ks][1]);
    p[ks][1] = pack_bf16(s[2 * ks][2], s[2 * ks][3]);
    p[ks][2] = pack_bf16(s[2 * ks + 1][0], s[2 * ks + 1][1]);
    p[ks][3] = pack_bf16(s[2 * ks + 1][2], s[2 * ks + 1][3]);
  }
}

__device__ __forceinline__ float quad_max(float v) {
  v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 1));
  return fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 2));
}
__device__ __forceinline__ float quad_sum(float v) {
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  return v + __shfl_xor_sync(0xffffffffu, v, 2);
}

// ============================================================================== forward
// CTA = 128 query rows (8 warps x 16 rows) of one (batch, head); key blocks of 64, double-buffered.
constexpr int FWD_BN = 64;

template <int FWD_BM>
__global__ void __launch_bounds__(FWD_BM * 2) attn_fwd_kernel(int T, int H, const bf16* __restrict__ qkv,
                                                              bf16* __restrict__ o, float* __restrict__ lse) {
  constexpr int FWD_THREADS = FWD_BM * 2;   // one warp per 16 query rows
  extern __shared__ __align__(128) uint8_t smem[];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int qb = (int)gridDim.x - 1 - (int)blockIdx.x;    // heaviest (last) query blocks first
  const int h = blockIdx.y, b = blockIdx.z;
  const int D = H * DH;
  const size_t ld = 3 * (size_t)D;
  const bf16* base = qkv + (size_t)b * T * ld + h * DH;
  const int q0 = qb * FWD_BM;
  const uint32_t sQ = smem_addr(smem), sK0 = sQ + FWD_BM * 128, sV0 = sK0 + 2 * FWD_BN * 128;
  const int n_kb = (q0 + FWD_BM) / FWD_BN;                 // causal: key blocks 0 .. n_kb-1

  load_tile<FWD_BM, FWD_THREADS>(sQ, base + (size_t)q0 * ld, ld, tid);
  load_tile<FWD_BN, FWD_THREADS>(sK0, base + D, ld, tid);
  load_tile<FWD_BN, FWD_THREADS>(sV0, base + 2 * D, ld, tid);
  cp_async_commit();

  const float c = rsqrtf((float)DH) * LOG2E;
  const int r0 = warp * 16;
  const int row_a = q0 + r0 + (lane >> 2), row_b = row_a + 8;   // the two query rows this thread owns
  float m_a = -INFINITY, m_b = -INFINITY, l_a = 0.f, l_b = 0.f;
  float oacc[8][4];
#pragma unroll
  for (int i = 0; i < 8; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) oacc[i][j] = 0.f;
  uint32_t qf[4][4];

  for (int kb = 0; kb < n_kb; ++kb) {
    const int buf = kb & 1;
    if (kb + 1 < n_kb) {   // prefetch the next key block into the other buffer
      load_tile<FWD_BN, FWD_THREADS>(sK0 + (buf ^ 1) * FWD_BN * 128, base + (size_t)(kb + 1) * FWD_BN * ld + D, ld, tid);
      load_tile<FWD_BN, FWD_THREADS>(sV0 + (buf ^ 1) * FWD_BN * 128, base + (size_t)(kb + 1) * FWD_BN * ld + 2 * D, ld, tid);
      cp_async_commit();
      cp_async_wait<1>();
    } else {
      cp_async_wait<0>();
    }
    __syncthreads();
    if (kb == 0) load_a_frags(qf, sQ, r0, lane);
    const int k0 = kb * FWD_BN;
    if (k0 <= q0 + r0) {        // warp-uniform: skip key blocks entirely above this warp's rows (k0, r0
                                // are multiples of 16, so every kept row sees at least key k0: no empty rows)
      float s[8][4];
#pragma unroll
      for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) s[i][j] = 0.f;
      mma_a_bT(s, qf, sK0 + buf * FWD_BN * 128, lane);
      const bool diag = k0 + FWD_BN - 1 > q0 + r0;          // some key of this block is masked for some row
      float mx_a = m_a, mx_b = m_b;
#pragma unroll
      for (int nt = 0; nt < 8; ++nt) {
        const int key = k0 + nt * 8 + (lane & 3) * 2;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const int kk = key + (j & 1), rr = (j < 2) ? row_a : row_b;
          s[nt][j] = (diag && kk > rr) ? -INFINITY : s[nt][j] * c;
        }
        mx_a = fmaxf(mx_a, fmaxf(s[nt][0], s[nt][1]));
        mx_b = fmaxf(mx_b, fmaxf(s[nt][2], s[nt][3]));
      }
      mx_a = quad_max(mx_a);
      mx_b = quad_max(mx_b);
      const float corr_a = exp2f(m_a - mx_a), corr_b = exp2f(m_b - mx_b);   // exp2(-inf) = 0 on the first block
      m_a = mx_a; m_b = mx_b;
      float sum_a = 0.f, sum_b = 0.f;
#pragma unroll
      for (int nt = 0; nt < 8; ++nt) {
        s[nt][0] = exp2f(s[nt][0] - m_a); s[nt][1] = exp2f(s[nt][1] - m_a);
        s[nt][2] = exp2f(s[nt][2] - m_b); s[nt][3] = exp2f(s[nt][3] - m_b);
        sum_a += s[nt][0] + s[nt][1];
        sum_b += s[nt][2] + s[nt][3];
      }
      l_a = l_a * corr_a + sum_a;
      l_b = l_b * corr_b + sum_b;
#pragma unroll
      for (int nt = 0; nt < 8; ++nt) {
        oacc[nt][0] *= corr_a; oacc[nt][1] *= corr_a;
        oacc[nt][2] *= corr_b; oacc[nt][3] *= corr_b;
      }
      uint32_t pf[4][4];
      acc_to_a(pf, s);
      mma_p_b(oacc, pf, sV0 + buf * FWD_BN * 128, lane);
    }
    __syncthreads();   // everyone is done with this buffer before the next prefetch overwrites it
  }
  l_a = quad_sum(l_a);
  l_b = quad_sum(l_b);
  const float inv_a = 1.f / l_a, inv_b = 1.f / l_b;
  bf16* oa = o + ((size_t)b * T + row_a) * D + h * DH + (lane & 3) * 2;
  bf16* ob = o + ((size_t)b * T + row_b) * D + h * DH + (lane & 3) * 2;
#pragma unroll
  for (int nt = 0; nt < 8; ++nt) {
    *reinterpret_cast<uint32_t*>(oa + nt * 8) = pack_bf16(oacc[nt][0] * inv_a, oacc[nt][1] * inv_a);
    *reinterpret_cast<uint32_t*>(ob + nt * 8) = pack_bf16(oacc[nt][2] * inv_b, oacc[nt][3] * inv_b);
  }
  if ((lane & 3) == 0) {
    float* L = lse + ((size_t)b * H + h) * T;
    L[row_a] = (m_a + log2f(l_a)) * LN2;
    L[row_b] = (m_b + log2f(l_b)) * LN2;
  }
}

// ============================================================================== backward
// delta[b,h,t] = sum_d do[b,t,h,d] * o[b,t,h,d]
__global__ void __launch_bounds__(256) attn_delta_kernel(size_t n_vec, int T, int H, const bf16* __restrict__ dout,
                                                         const bf16* __restrict__ o, float* __restrict__ delta) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;   // one 8-element vector per thread
  float acc = 0.f;
  if (i < n_vec) {
    float a[8], c[8];
    load_vec<bf16>(dout + i * 8, a);
    load_vec<bf16>(o + i * 8, c);
#pragma unroll
    for (int j = 0; j < 8; ++j) acc += a[j] * c[j];
  }
  acc += __shfl_xor_sync(0xffffffffu, acc, 1);
  acc += __shfl_xor_sync(0xffffffffu, acc, 2);
  acc += __shfl_xor_sync(0xffffffffu, acc, 4);
  if (i < n_vec && (threadIdx.x & 7) == 0) {
    const size_t hv = i >> 3;                 // (b*T + t)*H + h
    const int h = (int)(hv % H);
    const size_t bt = hv / H;
    const int t = (int)(bt % T);
    const size_t b = bt / T;
    delta[(b * H + h) * T + t] = acc;
  }
}

constexpr int BWD_B = 64, BWD_THREADS = 128;   // 64 x 64 blocks, 4 warps x 16 rows

// dK, dV of one 64-key block: rows = keys.  S^T = K Q^T, dP^T = V dO^T, dV += P^T dO, dK += dS^T Q.
__global__ void __launch_bounds__(BWD_THREADS) attn_bwd_dkdv_kernel(int T, int H, const bf16* __restrict__ dout,
                                                                    const bf16* __restrict__ qkv,
                                                                    const float* __restrict__ lse,
                                                                    const float* __restrict__ delta,
                                                                    bf16* __restrict__ dqkv) {
  extern __shared__ __align__(128) uint8_t smem[];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int jb = blockIdx.x, h = blockIdx.y, b = blockIdx.z;   // block 0 has the most work and starts first
  const int D = H * DH, n_qb = T / BWD_B;
  const size_t ld = 3 * (size_t)D;
  const bf16* base = qkv + (size_t)b * T * ld + h * DH;
  const bf16* dob = dout + (size_t)b * T * D + h * DH;
  const float* Lb = lse + ((size_t)b * H + h) * T;
  const float* Db = delta + ((size_t)b * H + h) * T;
  const uint32_t sK = smem_addr(smem), sV = sK + BWD_B * 128, sQ0 = sV + BWD_B * 128, sO0 = sQ0 + 2 * BWD_B * 128;
  float* sL = reinterpret_cast<float*>(smem + 6 * BWD_B * 128);   // [2][64] lse*log2e
  float* sD = sL + 2 * BWD_B;                                     // [2][64] delta
  const int k0 = jb * BWD_B;

  load_tile<BWD_B, BWD_THREADS>(sK, base + (size_t)k0 * ld + D, ld, tid);
  load_tile<BWD_B, BWD_THREADS>(sV, base + (size_t)k0 * ld + 2 * D, ld, tid);
  load_tile<BWD_B, BWD_THREADS>(sQ0, base + (size_t)k0 * ld, ld, tid);           // first query block = diagonal
  load_tile<BWD_B, BWD_THREADS>(sO0, dob + (size_t)k0 * D, D, tid);
  cp_async_commit();
  if (tid < BWD_B) { sL[tid] = Lb[k0 + tid] * LOG2E; sD[tid] = Db[k0 + tid]; }

  const float scale = rsqrtf((float)DH), c = scale * LOG2E;
  const int r0 = warp * 16;
  const int key_a = k0 + r0 + (lane >> 2), key_b = key_a + 8;
  float dk[8][4], dv[8][4];
#pragma unroll
  for (int i = 0; i < 8; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) dk[i][j] = dv[i][j] = 0.f;
  uint32_t kf[4][4], vf[4][4];

  for (int qb = jb; qb < n_qb; ++qb) {
    const int buf = (qb - jb) & 1;
    if (qb + 1 < n_qb) {
      const int qn = (qb + 1) * BWD_B;
      load_tile<BWD_B, BWD_THREADS>(sQ0 + (buf ^ 1) * BWD_B * 128, base + (size_t)qn * ld, ld, tid);
      load_tile<BWD_B, BWD_THREADS>(sO0 + (buf ^ 1) * BWD_B * 128, dob + (size_t)qn * D, D, tid);
      cp_async_commit();
      if (tid < BWD_B) { sL[(buf ^ 1) * BWD_B + tid] = Lb[qn + tid] * LOG2E; sD[(buf ^ 1) * BWD_B + tid] = Db[qn + tid]; }
      cp_async_wait<1>();
    } else {
      cp_async_wait<0>();
    }
    __syncthreads();
    if (qb == jb) { load_a_frags(kf, sK, r0, lane); load_a_frags(vf, sV, r0, lane); }
    const uint32_t sQ = sQ0 + buf * BWD_B * 128, sO = sO0 + buf * BWD_B * 128;
    const float* L = sL + buf * BWD_B;
    const float* Dl = sD + buf * BWD_B;
    float st[8][4], dp[8][4];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) st[i][j] = dp[i][j] = 0.f;
    mma_a_bT(st, kf, sQ, lane);    // S^T[key][query]
    mma_a_bT(dp, vf, sO, lane);    // dP^T[key][query]
    const int q0 = qb * BWD_B;
    const bool diag = qb == jb;
#pragma unroll
    for (int nt = 0; nt < 8; ++nt) {
      const int ql = nt * 8 + (lane & 3) * 2;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int qq = ql + (j & 1), key = (j < 2) ? key_a : key_b;
        float p = exp2f(st[nt][j] * c - L[qq]);
        if (diag && q0 + qq < key) p = 0.f;
        st[nt][j] = p;
        dp[nt][j] = p * (dp[nt][j] - Dl[qq]);
      }
    }
    uint32_t pf[4][4];
    acc_to_a(pf, st);
    mma_p_b(dv, pf, sO, lane);     // dV += P^T dO
    acc_to_a(pf, dp);
    mma_p_b(dk, pf, sQ, lane);     // dK += dS^T Q
    __syncthreads();
  }
  bf16* ka = dqkv + ((size_t)b * T + key_a) * ld + D + h * DH + (lane & 3) * 2;
  bf16* kb_ = dqkv + ((size_t)b * T + key_b) * ld + D + h * DH + (lane & 3) * 2;
#pragma unroll
  for (int nt = 0; nt < 8; ++nt) {
    *reinterpret_cast<uint32_t*>(ka + nt * 8) = pack_bf16(dk[nt][0] * scale, dk[nt][1] * scale);
    *reinterpret_cast<uint32_t*>(kb_ + nt * 8) = pack_bf16(dk[nt][2] * scale, dk[nt][3] * scale);
    *reinterpret_cast<uint32_t*>(ka + D + nt * 8) = pack_bf16(dv[nt][0], dv[nt][1]);
    *reinterpret_cast<uint32_t*>(kb_ + D + nt * 8) = pack_bf16(dv[nt][2], dv[nt][3]);
  }
}

// dQ of one 64-query block: S = Q K^T, dP = dO V^T, dQ += dS K.
__global__ void __launch_bounds__(BWD_THREADS) attn_bwd_dq_kernel(int T, int H, const bf16* __restrict__ dout,
                                                                  const bf16* __restrict__ qkv,
                                                                  const float* __restrict__ lse,
                                                                  const float* __restrict__ delta,
                                                                  bf16* __restrict__ dqkv) {
  extern __shared__ __align__(128) uint8_t smem[];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int qb = (int)gridDim.x - 1 - (int)blockIdx.x, h = blockIdx.y, b = blockIdx.z;
  const int D = H * DH;
  const size_t ld = 3 * (size_t)D;
  const bf16* base = qkv + (size_t)b * T * ld + h * DH;
  const bf16* dob = dout + (size_t)b * T * D + h * DH;
  const uint32_t sQ = smem_addr(smem), sO = sQ + BWD_B * 128, sK0 = sO + BWD_B * 128, sV0 = sK0 + 2 * BWD_B * 128;
  const int q0 = qb * BWD_B;

  load_tile<BWD_B, BWD_THREADS>(sQ, base + (size_t)q0 * ld, ld, tid);
  load_tile<BWD_B, BWD_THREADS>(sO, dob + (size_t)q0 * D, D, tid);
  load_tile<BWD_B, BWD_THREADS>(sK0, base + D, ld, tid);
  load_tile<BWD_B, BWD_THREADS>(sV0, base + 2 * D, ld, tid);
  cp_async_commit();

  const float scale = rsqrtf((float)DH), c = scale * LOG2E;
  const int r0 = warp * 16;
  const int row_a = q0 + r0 + (lane >> 2), row_b = row_a + 8;
  const float* Lb = lse + ((size_t)b * H + h) * T;
  const float* Db = delta + ((size_t)b * H + h) * T;
  const float L_a = Lb[row_a] * LOG2E, L_b = Lb[row_b] * LOG2E, D_a = Db[row_a], D_b = Db[row_b];
  float dq[8][4];
#pragma unroll
  for (int i = 0; i < 8; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) dq[i][j] = 0.f;
  uint32_t qf[4][4], of[4][4];

  for (int kb = 0; kb <= qb; ++kb) {
    const int buf = kb & 1;
    if (kb + 1 <= qb) {
      load_tile<BWD_B, BWD_THREADS>(sK0 + (buf ^ 1) * BWD_B * 128, base + (size_t)(kb + 1) * BWD_B * ld + D, ld, tid);
      load_tile<BWD_B, BWD_THREADS>(sV0 + (buf ^ 1) * BWD_B * 128, base + (size_t)(kb + 1) * BWD_B * ld + 2 * D, ld, tid);
      cp_async_commit();
      cp_async_wait<1>();
    } else {
      cp_async_wait<0>();
    }
    __syncthreads();
    if (kb == 0) { load_a_frags(qf, sQ, r0, lane); load_a_frags(of, sO, r0, lane); }
    const uint32_t sK = sK0 + buf * BWD_B * 128, sV = sV0 + buf * BWD_B * 128;
    float s[8][4], dp[8][4];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) s[i][j] = dp[i][j] = 0.f;
    mma_a_bT(s, qf, sK, lane);
    mma_a_bT(dp, of, sV, lane);
    const int k0 = kb * BWD_B;
    const bool diag = kb == qb;
#pragma unroll
    for (int nt = 0; nt < 8; ++nt) {
      const int key = k0 + nt * 8 + (lane & 3) * 2;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int kk = key + (j & 1);
        const bool top = j < 2;
        float p = exp2f(s[nt][j] * c - (top ? L_a : L_b));
        if (diag && kk > (top ? row_a : row_b)) p = 0.f;
        dp[nt][j] = p * (dp[nt][j] - (top ? D_a : D_b));
      }
    }
    uint32_t pf[4][4];
    acc_to_a(pf, dp);
    mma_p_b(dq, pf, sK, lane);     // dQ += dS K
    __syncthreads();
  }
  bf16* qa = dqkv + ((size_t)b * T + row_a) * ld + h * DH + (lane & 3) * 2;
  bf16* qb_ = dqkv + ((size_t)b * T + row_b) * ld + h * DH + (lane & 3) * 2;
#pragma unroll
  for (int nt = 0; nt < 8; ++nt) {
    *reinterpret_cast<uint32_t*>(qa + nt * 8) = pack_bf16(dq[nt][0] * scale, dq[nt][1] * scale);
    *reinterpret_cast<uint32_t*>(qb_ + nt * 8) = pack_bf16(dq[nt][2] * scale, dq[nt][3] * scale);
  }
}

}  // namespace

int attention_fwd_mma(int mu, int T, int H, const void* qkv, void* o, float* lse, cudaStream_t s) {
  static bool set = false;
  if (!set) {
    PACI_CUDA_OK(cudaFuncSetAttribute(attn_fwd_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      128 * 128 + 4 * FWD_BN * 128));
    set = true;
  }
  if (T % 128 == 0) {   // 128-query CTAs (8 warps); T is a multiple of 64 (validated by the caller)
    dim3 grid(T / 128, H, mu);
    PACI_LAUNCH(attn_fwd_kernel<128>, grid, 256, 128 * 128 + 4 * FWD_BN * 128, s, T, H, (const bf16*)qkv, (bf16*)o, lse);
  } else {
    dim3 grid(T / 64, H, mu);
    PACI_LAUNCH(attn_fwd_kernel<64>, grid, 128, 64 * 128 + 4 * FWD_BN * 128, s, T, H, (const bf16*)qkv, (bf16*)o, lse);
  }
  return PACI_OK;
}

size_t attention_bwd_mma_scratch_bytes(int mu, int T, int H) { return (size_t)mu * H * T * sizeof(float); }

int attention_bwd_mma(int mu, int T, int H, const void* dout, const void* qkv, const void* o, const float* lse,
                      void* dqkv, float* scratch, cudaStream_t s) {
  const size_t n_vec = (size_t)mu * T * H * DH / 8;
  PACI_LAUNCH(attn_delta_kernel, ceil_div(n_vec, 256), 256, 0, s, n_vec, T, H, (const bf16*)dout, (const bf16*)o,
              scratch);
  constexpr int SMEM1 = 6 * BWD_B * 128 + 4 * BWD_B * 4, SMEM2 = 6 * BWD_B * 128;
  static bool set = false;
  if (!set) {
    PACI_CUDA_OK(cudaFuncSetAttribute(attn_bwd_dkdv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM1));
    PACI_CUDA_OK(cudaFuncSetAttribute(attn_bwd_dq_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM2));
    set = true;
  }
  dim3 grid(T / BWD_B, H, mu);
  PACI_LAUNCH(attn_bwd_dkdv_kernel, grid, BWD_THREADS, SMEM1, s, T, H, (const bf16*)dout, (const bf16*)qkv, lse,
              scratch, (bf16*)dqkv);
  PACI_LAUNCH(attn_bwd_dq_kernel, grid, BWD_THREADS, SMEM2, s, T, H, (const bf16*)dout, (const bf16*)qkv, lse,
              scratch, (bf16*)dqkv);
  return PACI_OK;
}

}  // namespace paci
