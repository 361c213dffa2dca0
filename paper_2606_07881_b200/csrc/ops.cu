// ops.cu -- dispatch on the stage's dtype (PACI_FP32 -> the FFMA parity kernels, PACI_BF16 -> the tcgen05 kernels;
// one kernel family per dtype, no switches) and the
// op-level C-ABI entry points used by the kernel parity tests and the per-kernel roofline benches.
#include <algorithm>
#include <cstdlib>
#include <cstring>

#include "common.cuh"

namespace paci {

int gemm(int dtype, int layout, int M, int N, int K, const void* A, int lda, const void* B, int ldb,
         const float* bias, void* C, int ldc, int out_f32_accum, cudaStream_t s) {
  if (M <= 0 || N <= 0) return PACI_OK;                 // empty output
  if (K <= 0) {                                         // empty contraction: nothing to add; an overwrite has no value
    if (out_f32_accum) return PACI_OK;
    return fail(PACI_EINVAL, "gemm: K = %d with an overwritten output", K);
  }
  const double e = dtype == PACI_BF16 ? 2.0 : 4.0;
  ProfScope prof(layout == 0 ? PC_GEMM_FWD : layout == 1 ? PC_GEMM_DGRAD : PC_GEMM_WGRAD, 2.0 * M * N * K,
                 e * ((double)M * K + (double)N * K) + (out_f32_accum ? 8.0 : e) * M * N, s);
  if (dtype == PACI_BF16)
    return gemm_tc(layout, M, N, K, A, lda, B, ldb, bias, C, ldc, out_f32_accum, s);
  return gemm_simt(dtype, layout, M, N, K, A, lda, B, ldb, bias, C, ldc, out_f32_accum, s);
}

int gemm_backward_pair(int dtype, int M, int N_out, int K_in, const void* dy, int ld_dy, const void* x, int ld_x,
                       const void* W, int ld_w, float* G_W, int ld_g, void* dx, int ld_dx, cudaStream_t s) {
  if (M <= 0 || N_out <= 0 || K_in <= 0) return PACI_OK;   // no tokens: dx is empty and G_W gets nothing
  if (dtype == PACI_BF16) {
    ProfScope prof(PC_GEMM_BWD_PAIR, 4.0 * M * (double)N_out * K_in,
                   2.0 * (2.0 * (double)M * N_out + (double)M * K_in + (double)N_out * K_in) + 8.0 * N_out * K_in + 2.0 * M * K_in, s);
    const GemmDesc d[2] = {
        {2, N_out, K_in, M, dy, ld_dy, x, ld_x, nullptr, G_W, ld_g, 1, nullptr},      // G_W += dy^T x
        {1, M, K_in, N_out, dy, ld_dy, W, ld_w, nullptr, dx, ld_dx, 0, nullptr}};     // dx = dy W
    return gemm_tc_multi(d, 2, s);
  }
  int rc = gemm(dtype, 1, M, K_in, N_out, dy, ld_dy, W, ld_w, nullptr, dx, ld_dx, 0, s);
  if (rc != PACI_OK) return rc;
  return gemm(dtype, 2, N_out, K_in, M, dy, ld_dy, x, ld_x, nullptr, G_W, ld_g, 1, s);
}

// Backward of the attention output projection y = o Wo^T (rows a16 + the prologue of a17): G_Wo += dy^T o and
// d_o = dy Wo in one launch; on the tcgen05 path the dgrad's epilogue also leaves delta = rowsum(d_o * o) per head and
// lse log2(e) in `attn_scratch` (the layout attention_bwd_tc reads), *prepared = 1, and attention_bwd is then called
// with scratch_prepared = 1 and launches no delta kernel.  Otherwise *prepared = 0 and nothing else changes.
int out_proj_backward(int dtype, int mu, int T, int H, int dh, const void* dy, const void* o, const void* Wo,
                      float* G_Wo, void* d_o, const float* lse, float* attn_scratch, int* prepared, cudaStream_t s) {
  const int M = mu * T, D = H * dh;
  *prepared = 0;
  if (dtype == PACI_BF16 && dh == 64 && T % 128 == 0 && mu > 0 && lse != nullptr && attn_scratch != nullptr) {
    ProfScope prof(PC_GEMM_BWD_PAIR, 4.0 * M * (double)D * D,
                   2.0 * (2.0 * (double)M * D + (double)M * D + (double)D * D) + 8.0 * D * D + 2.0 * M * D, s);
    const AttnDeltaOut a{o, D, lse, attn_scratch, attn_scratch + (size_t)mu * H * T, T, H};
    const GemmDesc d[2] = {
        {2, D, D, M, dy, D, o, D, nullptr, G_Wo, D, 1, nullptr, nullptr},       // G_Wo += dy^T o
        {1, M, D, D, dy, D, Wo, D, nullptr, d_o, D, 0, nullptr, &a}};           // d_o = dy Wo (+ delta, lse2)
    *prepared = 1;
    return gemm_tc_multi(d, 2, s);
  }
  return gemm_backward_pair(dtype, M, D, D, dy, D, o, D, Wo, D, G_Wo, D, d_o, D, s);
}

int gemm_bias_gelu(int dtype, int M, int N, int K, const void* A, int lda, const void* B, int ldb, const float* bias,
                   void* C, void* Gout, int ldc, cudaStream_t s) {
  if (M <= 0 || N <= 0) return PACI_OK;
  if (K <= 0) return fail(PACI_EINVAL, "gemm_bias_gelu: K = %d", K);
  if (dtype == PACI_BF16) {
    ProfScope prof(PC_GEMM_FWD, 2.0 * M * N * K, 2.0 * ((double)M * K + (double)N * K) + 4.0 * M * N, s);
    return gemm_tc(0, M, N, K, A, lda, B, ldb, bias, C, ldc, 0, s, Gout);
  }
  int rc = gemm(dtype, 0, M, N, K, A, lda, B, ldb, bias, C, ldc, 0, s);
  if (rc != PACI_OK) return rc;
  if (ldc != N) return fail(PACI_EINVAL, "gemm_bias_gelu: the unfused path needs ldc == N");
  return gelu_fwd(dtype, (size_t)M * N, C, Gout, s);
}

int attention_fwd_tc(int mu, int T, int H, const void* qkv, void* o, float* lse, cudaStream_t s);
int attention_bwd_tc(int mu, int T, int H, const void* dout, const void* qkv, const void* o, const float* lse,
                     void* dqkv, float* scratch, float* Gbias, int scratch_prepared, cudaStream_t s);
size_t attention_bwd_tc_scratch_bytes(int mu, int T, int H);

// algorithmic work: causal half of QK^T and PV (2 * mu*H*T*T*dh flops forward, twice that backward)
int attention_fwd(int dtype, int mu, int T, int H, int dh, const void* qkv, void* o, float* lse, cudaStream_t s) {
  const double e = dtype == PACI_BF16 ? 2.0 : 4.0, nd = (double)mu * T * H * dh;
  ProfScope prof(PC_ATTN_FWD, 2.0 * mu * H * (double)T * T * dh, e * 4.0 * nd + 4.0 * mu * H * T, s);
  if (dtype == PACI_BF16) {
    if (dh != 64 || T % 128) return fail(PACI_EINVAL, "bf16 attention needs head dim 64 and T %% 128 == 0");
    return attention_fwd_tc(mu, T, H, qkv, o, lse, s);
  }
  return attention_fwd_simt(dtype, mu, T, H, dh, qkv, o, lse, s);
}

// Gbias (fp32 [3 H dh], may be NULL) += column sums of dqkv: the QKV bias gradient (row a15).  The tcgen05
// kernels take it in their epilogue; the fp32 parity kernels run the column-sum kernel over dqkv afterwards.
int attention_bwd(int dtype, int mu, int T, int H, int dh, const void* dout, const void* qkv, const void* o,
                  const float* lse, void* dqkv, float* scratch, float* Gbias, cudaStream_t s, int scratch_prepared) {
  int rc;
  {
    const double e = dtype == PACI_BF16 ? 2.0 : 4.0, nd = (double)mu * T * H * dh;
    ProfScope prof(PC_ATTN_BWD, 4.0 * mu * H * (double)T * T * dh, e * 8.0 * nd + 4.0 * mu * H * T, s);
    if (dtype == PACI_BF16) {
      if (dh != 64 || T % 128) return fail(PACI_EINVAL, "bf16 attention needs head dim 64 and T %% 128 == 0");
      return attention_bwd_tc(mu, T, H, dout, qkv, o, lse, dqkv, scratch, Gbias, scratch_prepared, s);
    }
    rc = attention_bwd_simt(dtype, mu, T, H, dh, dout, qkv, o, lse, dqkv, scratch, s);
  }
  if (rc == PACI_OK && Gbias != nullptr) rc = colsum(dtype, mu * T, 3 * H * dh, dqkv, Gbias, s);
  return rc;
}

size_t attention_bwd_scratch_bytes(int dtype, int mu, int T, int H, int dh) {
  const size_t simt = (size_t)mu * H * T * sizeof(float);
  if (dtype == PACI_BF16 && dh == 64) return std::max(simt, attention_bwd_tc_scratch_bytes(mu, T, H));
  return simt;
}

}  // namespace paci

using namespace paci;

extern "C" {

int paci_op_gemm(int dtype, int layout, int M, int N, int K, const void* A, int lda, const void* B, int ldb,
                 const float* bias, void* C, int ldc, int out_f32_accum, void* stream) {
  return gemm(dtype, layout, M, N, K, A, lda, B, ldb, bias, C, ldc, out_f32_accum, (cudaStream_t)stream);
}
int paci_op_gemm_backward_pair(int dtype, int M, int N_out, int K_in, const void* dy, int ld_dy, const void* x, int ld_x,
                               const void* W, int ld_w, float* G_W, int ld_g, void* dx, int ld_dx, void* stream) {
  return gemm_backward_pair(dtype, M, N_out, K_in, dy, ld_dy, x, ld_x, W, ld_w, G_W, ld_g, dx, ld_dx, (cudaStream_t)stream);
}
int paci_op_gemm_bias_gelu(int dtype, int M, int N, int K, const void* A, int lda, const void* B, int ldb,
                           const float* bias, void* C, void* G, int ldc, void* stream) {
  return gemm_bias_gelu(dtype, M, N, K, A, lda, B, ldb, bias, C, G, ldc, (cudaStream_t)stream);
}
int paci_op_layernorm_fwd(int dtype, int rows, int D, const void* x, const void* res, const float* g,
                          const float* b, void* xsum, void* y, float* mean, float* rstd, void* stream) {
  return ln_fwd(dtype, rows, D, x, res, g, b, xsum, y, mean, rstd, (cudaStream_t)stream);
}
int paci_op_layernorm_bwd(int dtype, int rows, int D, const void* dy, const void* x, const float* mean,
                          const float* rstd, const float* g, const void* dres, void* dx, float* Gg, float* Gb,
                          float* Gcol, void* stream) {
  return ln_bwd(dtype, rows, D, dy, x, mean, rstd, g, dres, dx, Gg, Gb, Gcol, (cudaStream_t)stream);
}
int paci_op_gelu_fwd(int dtype, size_t n, const void* p, void* out, void* stream) {
  return gelu_fwd(dtype, n, p, out, (cudaStream_t)stream);
}
int paci_op_gelu_bwd(int dtype, int rows, int cols, const void* dg, const void* p, void* dp, float* Gbias,
                     void* stream) {
  return gelu_bwd(dtype, rows, cols, dg, p, dp, Gbias, (cudaStream_t)stream);
}
int paci_op_colsum(int dtype, int rows, int cols, const void* x, float* G, void* stream) {
  return colsum(dtype, rows, cols, x, G, (cudaStream_t)stream);
}
int paci_op_attention_fwd(int dtype, int mu, int T, int H, int dh, const void* qkv, void* o, float* lse,
                          void* stream) {
  return attention_fwd(dtype, mu, T, H, dh, qkv, o, lse, (cudaStream_t)stream);
}
int paci_op_out_proj_backward(int dtype, int mu, int T, int H, int dh, const void* dy, const void* o, const void* Wo,
                              float* G_Wo, void* d_o, const float* lse, float* attn_scratch, int* prepared, void* stream) {
  if (prepared == nullptr) return fail(PACI_EINVAL, "paci_op_out_proj_backward: prepared is NULL");
  return out_proj_backward(dtype, mu, T, H, dh, dy, o, Wo, G_Wo, d_o, lse, attn_scratch, prepared, (cudaStream_t)stream);
}
int paci_op_attention_bwd_prepared(int dtype, int mu, int T, int H, int dh, const void* dout, const void* qkv,
                                   const void* o, const float* lse, void* dqkv, float* scratch, void* stream) {
  return attention_bwd(dtype, mu, T, H, dh, dout, qkv, o, lse, dqkv, scratch, nullptr, (cudaStream_t)stream, 1);
}
int paci_op_attention_bwd(int dtype, int mu, int T, int H, int dh, const void* dout, const void* qkv,
                          const void* o, const float* lse, void* dqkv, float* scratch, void* stream) {
  return attention_bwd(dtype, mu, T, H, dh, dout, qkv, o, lse, dqkv, scratch, nullptr, (cudaStream_t)stream);
}
size_t paci_op_attention_bwd_scratch_bytes(int dtype, int mu, int T, int H, int dh) {
  return attention_bwd_scratch_bytes(dtype, mu, T, H, dh);
}
int paci_op_embed_fwd(int dtype, int mu, int T, int D, int vocab, const int32_t* tok, const float* wte,
                      const float* wpe, void* x, void* stream) {
  return embed_fwd(dtype, mu, T, D, tok, wte, wpe, x, vocab, nullptr, (cudaStream_t)stream);
}
int paci_op_embed_bwd(int dtype, int mu, int T, int D, int vocab, const int32_t* tok, const void* dx, float* Gwte,
                      float* Gwpe, void* stream) {
  return embed_bwd(dtype, mu, T, D, tok, dx, Gwte, Gwpe, vocab, (cudaStream_t)stream);
}
int paci_op_softmax_ce(int dtype, int rows, int V, int ldz, void* z, const int32_t* tgt, float* loss,
                       void* stream) {
  return softmax_ce(dtype, rows, V, ldz, z, tgt, loss, nullptr, (cudaStream_t)stream);
}
int paci_op_dropout(int dtype, size_t n, const void* x, void* out, float p, uint64_t seed, int64_t mb_id,
                    int32_t site, void* stream) {
  return dropout(dtype, n, x, out, p, seed, mb_id, site, (cudaStream_t)stream);
}
int paci_op_adamw(size_t n, size_t n_decay, float* w, float* m, float* v, float* G, void* shadow_bf16, int k,
                  int64_t t, float lr, float beta1, float beta2, float eps, float weight_decay,
                  int64_t* version_word, void* stream) {
  return adamw(n, n_decay, w, m, v, G, shadow_bf16, k, t, lr, beta1, beta2, eps, weight_decay, version_word,
               (cudaStream_t)stream);
}

}  // extern "C"
