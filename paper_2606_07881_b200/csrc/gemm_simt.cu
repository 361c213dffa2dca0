// gemm_simt.cu -- plain FFMA GEMM.  This IS the product path in PACI_FP32 mode (the 1e-5 parity
// mode of the tiny config: tcgen05 kind::tf32 cannot meet 1e-5), and it serves shapes the tcgen05
// kernel does not take (ragged tiny shapes).  In PACI_BF16 mode it is used only when the environment
// variable PACI_GEMM=simt forces it (debugging aid) -- never silently.
//
// C(m,n) = sum_k A(m,k) * B(n,k), operands addressed through (row, k) strides so that the three
// layouts of paci_op_gemm (NT forward, NN dgrad, TN wgrad) share one kernel.
#include "common.cuh"

namespace paci {

template <typename T>
__global__ void __launch_bounds__(256) gemm_simt_kernel(int M, int N, int K, const T* __restrict__ A, long a_sm,
                                                        long a_sk, const T* __restrict__ B, long b_sn, long b_sk,
                                                        const float* __restrict__ bias, void* __restrict__ Cv,
                                                        int ldc, int accum) {
  PACI_PDL_SYNC;
  constexpr int BM = 64, BN = 64, BK = 16;
  __shared__ float As[BK][BM + 4];
  __shared__ float Bs[BK][BN + 4];
  const int tx = threadIdx.x % 16, ty = threadIdx.x / 16;
  const int m0 = blockIdx.y * BM, n0 = blockIdx.x * BN;
  float acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;

  for (int k0 = 0; k0 < K; k0 += BK) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int idx = threadIdx.x + 256 * i;
      int mm, kk;
      if (a_sk == 1) { kk = idx % BK; mm = idx / BK; } else { mm = idx % BM; kk = idx / BM; }
      const int gm = m0 + mm, gk = k0 + kk;
      As[kk][mm] = (gm < M && gk < K) ? to_f(A[(long)gm * a_sm + (long)gk * a_sk]) : 0.f;
      int nn;
      if (b_sk == 1) { kk = idx % BK; nn = idx / BK; } else { nn = idx % BN; kk = idx / BN; }
      const int gn = n0 + nn;
      const int gk2 = k0 + kk;
      Bs[kk][nn] = (gn < N && gk2 < K) ? to_f(B[(long)gn * b_sn + (long)gk2 * b_sk]) : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < BK; ++kk) {
      float a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = As[kk][ty * 4 + i];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = Bs[kk][tx * 4 + j];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int gm = m0 + ty * 4 + i;
    if (gm >= M) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int gn = n0 + tx * 4 + j;
      if (gn >= N) continue;
      if (accum) {
        float* C = reinterpret_cast<float*>(Cv);
        C[(size_t)gm * ldc + gn] += acc[i][j];      // beta = 1 (Alg. 1 line 13); one owner per element
      } else {
        T* C = reinterpret_cast<T*>(Cv);
        C[(size_t)gm * ldc + gn] = from_f<T>(acc[i][j] + (bias != nullptr ? bias[gn] : 0.f));
      }
    }
  }
}

int gemm_simt(int dtype, int layout, int M, int N, int K, const void* A, int lda, const void* B, int ldb,
              const float* bias, void* C, int ldc, int out_f32_accum, cudaStream_t s) {
  if (M <= 0 || N <= 0) return PACI_OK;
  long a_sm, a_sk, b_sn, b_sk;
  switch (layout) {
    case 0: a_sm = lda; a_sk = 1; b_sn = ldb; b_sk = 1; break;   // NT: A[M,K], B[N,K]
    case 1: a_sm = lda; a_sk = 1; b_sn = 1; b_sk = ldb; break;   // NN: A[M,K], B[K,N]
    case 2: a_sm = 1; a_sk = lda; b_sn = 1; b_sk = ldb; break;   // TN: A[K,M], B[K,N]
    default: return fail(PACI_EINVAL, "gemm: layout %d", layout);
  }
  dim3 grid(ceil_div(N, 64), ceil_div(M, 64));
  if (dtype == PACI_BF16)
    PACI_LAUNCH(gemm_simt_kernel<bf16>, grid, 256, 0, s, M, N, K, (const bf16*)A, a_sm, a_sk, (const bf16*)B, b_sn,
                b_sk, bias, C, ldc, out_f32_accum);
  else
    PACI_LAUNCH(gemm_simt_kernel<float>, grid, 256, 0, s, M, N, K, (const float*)A, a_sm, a_sk, (const float*)B,
                b_sn, b_sk, bias, C, ldc, out_f32_accum);
  return PACI_OK;
}

}  // namespace paci
