/* paci.h -- C ABI of the B200-native PACI stage-step library (libpaci.so).
 *
 * PACI = Pipeline Asynchronous training with Controlled Inconsistency
 * (/root/reference/PAPER.md; "P:n" below = line n of that file).
 *
 * The library implements the per-stage micro-batch step of Algorithm 1:
 *   forward  F_i(h_{m,i-1}; theta_i)                       (Eq. 7; Alg. 1 lines 5-9)
 *   backward g_{m,i}, grad h_{m,i-1} with the activations stashed at forward time and the
 *            stage's CURRENT parameters                    (Eq. 1; Alg. 1 lines 11-15)
 *   G_i += g_{m,i} in place, in fp32                        (Alg. 1 line 13)
 *   one fused AdamW update every k local backwards          (Alg. 1 lines 16-19)
 * under a per-stage parameter-version counter t and the admission rule q_i <= N-i
 * (Eq. 9), and reports for every micro-batch the number of updates that fell between its
 * forward and its backward, Delta_{m,i} = t^B - t^F (Eq. 8).
 *
 * Conventions
 *   - plain C, no torch types.  Every pointer says HOST or DEVICE.  Sizes are in elements unless
 *     they end in _bytes.  `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *   - the library allocates NO device memory and creates NO streams for a stage: the caller owns
 *     the workspace and every in/out buffer and must keep them alive until the enqueued work is done.
 *   - all compute calls are asynchronous on `stream`; host counters advance at enqueue time, and the
 *     per-stage stream order equals the call order, so host-side Delta equals device-side Delta.
 *     A device-side stamp (a version word bumped by the AdamW kernel and sampled by the first kernel
 *     of every forward/backward) is kept so that tests can prove it (paci_stage_device_stamps).
 *   - return value: 0 (PACI_OK) or a negative error code; never throws.  paci_last_error() returns
 *     a thread-local human-readable message for the last failing call.
 *   - activations are row-major [mu, T, D] in the stage's compute dtype (float for PACI_FP32,
 *     __nv_bfloat16 for PACI_BF16); tokens/targets are int32 [mu, T].
 *   - stage_index s is 0-based; the paper's stage i is s+1, its N is n_stages, its a is k_accum.
 *   - one kernel family per dtype (PACI_FP32: FFMA parity kernels; PACI_BF16: tcgen05 / TMA kernels); no
 *     environment switches, no fallback paths.
 */
#ifndef PACI_H_
#define PACI_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- error codes ------------------------------------------------------------------------ */
#define PACI_OK       0
#define PACI_EINVAL  (-1)  /* bad config / null or misaligned pointer / workspace too small          */
#define PACI_EAGAIN  (-2)  /* admission rule refuses the forward: q_s > S-1-s (Alg. 1 line 5).       */
                           /* State unchanged; retry after a backward.                               */
#define PACI_ESTATE  (-3)  /* call out of protocol: backward for a micro-batch that is not the        */
                           /* oldest unresolved forward (FIFO, R4); forward/backward while  */
                           /* an update is pending (c == k and paci_maybe_step not yet called);       */
                           /* mb_id reuse while unresolved.                                           */
#define PACI_ECUDA   (-4)  /* CUDA error at launch; text in paci_last_error()                        */

/* ---- dtypes ------------------------------------------------------------------------------ */
#define PACI_FP32 0        /* fp32 activations, weights, FFMA GEMMs (parity mode, 1e-5)             */
#define PACI_BF16 1        /* bf16 activations + bf16 weight shadow, tcgen05 GEMMs with fp32          */
                           /* accumulation; fp32 master weights, m, v, G; fp32 LN/softmax statistics */

/* ---- tensor groups for load/read ---------------------------------------------------------- */
#define PACI_PARAM      0  /* fp32 master parameters theta_i                                        */
#define PACI_GRAD_ACCUM 1  /* G_i: raw SUM of the window's gradients (the 1/k is applied in AdamW)    */
#define PACI_ADAM_M     2
#define PACI_ADAM_V     3

typedef struct paci_stage paci_stage_t;       /* opaque host object */

typedef struct paci_stage_config {
  int32_t stage_index;   /* s, 0-based                                                            */
  int32_t n_stages;      /* S (paper N).  Unresolved forwards allowed before admission: S-1-s     */
  int32_t n_layers;      /* pre-LN GPT-2 decoder blocks on this stage (>= 0)                      */
  int32_t d_model;       /* D, multiple of 8 (bf16: multiple of 64)                                */
  int32_t n_heads;       /* H, D % H == 0; head dim 64 in PACI_BF16, any <= 128 in PACI_FP32      */
  int32_t seq_len;       /* T (bf16: multiple of 128)                                              */
  int32_t micro_batch;   /* mu sequences per micro-batch; M = mu*T tokens                          */
  int32_t k_accum;       /* k (paper a): local backwards per optimizer update                      */
  int32_t vocab;         /* V (used when has_embedding or has_head)                                */
  int32_t has_embedding; /* stage holds wte, wpe and takes int32 tokens as input           */
  int32_t has_head;      /* stage holds final LN + LM head + mean token cross-entropy.     */
                         /* With has_embedding too the head is TIED to wte (one tensor, summed      */
                         /* gradient); otherwise the stage owns its own copy "head.w" (DESIGN R10)  */
  int32_t dtype;         /* PACI_FP32 | PACI_BF16                                                  */
  float beta1, beta2, eps, weight_decay;   /* AdamW: 0.9, 0.95, 1e-8, 0.1 in the paper    */
  int32_t checkpoint;    /* 0: backward differentiates the activations STASHED at forward time and  */
                         /*    evaluates them at the current parameters (Eq. 1).              */
                         /* 1: activation-checkpointed PACI (App. B "Activation checkpointing",     */
                         /*    P:282): only the stage INPUT (tokens / h, and the targets) is kept;  */
                         /*    backward first recomputes the stage forward under the stage's        */
                         /*    CURRENT parameter version, then differentiates that.  Same single    */
                         /*    parameter copy; a stash slot shrinks to the stage input.             */
  float   dropout_p;     /* dropout probability (0.1) on the embedding output and on the     */
                         /* output of both residual branches of every block (R23); 0 = off */
  uint64_t dropout_seed; /* key of the counter-based mask generator (Philox4x32-10, counter =       */
                         /* (mb_id, site, element/4)); backward regenerates the forward's mask      */
} paci_stage_config;

/* Bytes of DEVICE workspace a stage with this config needs (parameters, m, v, G, bf16 shadow,
 * S-s stash slots, scratch).  0 = invalid config (see paci_last_error). */
size_t paci_stage_workspace_bytes(const paci_stage_config* cfg);

/* Number of fp32 parameters of the stage (sum over tensors). 0 = invalid config. */
size_t paci_stage_param_count(const paci_stage_config* cfg);

/* Create a stage on the current CUDA device.  dev_ws: DEVICE, 256-byte aligned, >= workspace_bytes;
 * borrowed until paci_stage_destroy.  Zeroes m, v, G and the counters on `stream`; parameters are
 * undefined until paci_stage_load(PACI_PARAM, ...) has been called for every tensor. */
int paci_stage_create(const paci_stage_config* cfg, void* dev_ws, size_t ws_bytes, void* stream,
                      paci_stage_t** out);
int paci_stage_destroy(paci_stage_t* st);

/* Tensor names (stage-local): wte, wpe, h.<l>.ln1.g|b, h.<l>.attn.wqkv|bqkv|wo|bo, h.<l>.ln2.g|b,
 * h.<l>.mlp.w1|b1|w2|b2, lnf.g|b, head.w (only when has_head && !has_embedding).
 * Matrices are [out, in] row-major; wqkv rows are [q; k; v], head h = rows h*dh..(h+1)*dh-1 (R17).
 * Returns the element count, or 0 if the stage has no such tensor. */
size_t paci_stage_tensor_numel(const paci_stage_t* st, const char* name);

/* Copy a HOST fp32 array of n elements into / out of one tensor of group `what`.
 * load(PACI_PARAM) also refreshes the bf16 shadow.  Both synchronise `stream` before returning. */
int paci_stage_load(paci_stage_t* st, int what, const char* name, const float* host_src, size_t n,
                    void* stream);
int paci_stage_read(paci_stage_t* st, int what, const char* name, float* host_dst, size_t n,
                    void* stream);

/* Forward of micro-batch mb_id (Alg. 1 lines 5-9).
 *   in      DEVICE: int32 tokens [mu,T] if has_embedding, else h [mu,T,D] (compute dtype)
 *   targets DEVICE: int32 [mu,T] if has_head, else NULL
 *   out     DEVICE: h [mu,T,D] (compute dtype), or float loss[1] if has_head
 * Admission: refused with PACI_EAGAIN when q_s > S-1-s.  On success records t^F = version, takes a
 * stash slot, q_s += 1. */
int paci_forward(paci_stage_t* st, int64_t mb_id, const void* in, const int32_t* targets, void* out,
                 void* stream);
/* The same with n_seq <= micro_batch sequences in this micro-batch (heterogeneous micro-batch sizes,
 * App. B "Micro-batching": "the first B mod m micro-batches contain floor(B/m)+1 sequences and the
 * remaining micro-batches contain floor(B/m) sequences").  in / targets / out hold n_seq sequences; the loss
 * is the mean over the n_seq*T tokens of THIS micro-batch (R22).  paci_backward of mb_id works on
 * the n_seq recorded here. */
int paci_forward_var(paci_stage_t* st, int64_t mb_id, int32_t n_seq, const void* in, const int32_t* targets,
                     void* out, void* stream);

/* Backward of micro-batch mb_id (Alg. 1 lines 11-15): must be the oldest unresolved forward.
 *   dout DEVICE: grad wrt the stage output [mu,T,D] (compute dtype); NULL iff has_head
 *   din  DEVICE: grad wrt the stage input  [mu,T,D]; NULL iff has_embedding
 * Records Delta = version - t^F, accumulates weight gradients into G (fp32, in the GEMM epilogue),
 * c_s += 1, q_s -= 1, frees the stash slot. */
int paci_backward(paci_stage_t* st, int64_t mb_id, const void* dout, void* din, void* stream);

/* Alg. 1 lines 16-19: if c_s == k enqueue ONE fused multi-tensor AdamW kernel (update theta with
 * G/k and learning rate lr, refresh bf16 shadow, zero G, bump the device version word), then
 * version += 1, c_s = 0.  Returns 1 if it stepped, 0 if not yet, < 0 on error.  This is the only
 * call that changes parameters. */
int paci_maybe_step(paci_stage_t* st, float lr, void* stream);

/* Learning-rate schedule of App. B: linear warm-up over warmup_steps updates to `peak`, then cosine
 * decay to final_frac * peak at total_steps (paper: 1% warm-up, final_frac 0.1).  `step` = the stage's local
 * update index t (paci_version) BEFORE the update it is used for.  Pure host arithmetic (no device work):
 *   step <  warmup : peak * (step + 1) / warmup
 *   else           : peak * (f + (1 - f) * 0.5 * (1 + cos(pi * (step - warmup) / (total - warmup)))), clamped at
 *                    step >= total to peak * f.                                              (R16) */
float paci_lr_schedule(int64_t step, int64_t total_steps, int64_t warmup_steps, float peak, float final_frac);

/* Checkpoint / resume of the counters that paci_stage_load cannot reach: sets the local update index t
 * (also the AdamW bias-correction step and the DEVICE version word) and the window count c (0 <= c < k; the
 * matching partial sum must have been loaded into PACI_GRAD_ACCUM).  Only legal with no unresolved forward
 * (q = 0), else PACI_ESTATE.  Synchronises `stream`. */
int paci_stage_set_state(paci_stage_t* st, int64_t version, int32_t window_count, void* stream);
/* Device-side input validation: token / target ids outside [0, vocab) are CLAMPED by the kernels (never an
 * out-of-bounds access) and raise a sticky device flag.  Synchronises `stream`; returns PACI_EINVAL if the
 * flag is set (and clears it), else PACI_OK. */
int paci_stage_check(paci_stage_t* st, void* stream);

int64_t paci_version(const paci_stage_t* st);          /* local updates applied so far (t)       */
int32_t paci_unresolved(const paci_stage_t* st);       /* q_s                                          */
int32_t paci_window_count(const paci_stage_t* st);     /* c_s                                          */
/* Delta_{m,s} = t^B - t^F (Eq. 8) of a micro-batch whose backward has been enqueued;
 * -1 if unknown (never forwarded, or backward not yet called).  The log keeps the last 4096 ids. */
int32_t paci_crossed_updates(const paci_stage_t* st, int64_t mb_id);
/* Device-side proof of the same numbers: versions sampled ON THE DEVICE by the first kernel of the
 * forward and of the backward of mb_id.  Synchronises `stream`.  Returns 0 or PACI_EINVAL. */
int paci_stage_device_stamps(paci_stage_t* st, int64_t mb_id, int64_t* vF, int64_t* vB, void* stream);

const char* paci_last_error(void);

/* ---- schedule driver: S emulated stages on ONE GPU (BASELINE.json item 6) ------------------ */
#define PACI_MODE_PACI  0   /* asynchronous 1F1B + accumulation                         */
#define PACI_MODE_FLUSH 1   /* synchronous 1F1B-flush comparator; stages must have   */
                            /* been created with k_accum = m_f                                     */

typedef struct paci_pipeline paci_pipeline_t;

typedef struct paci_run_report {
  float*   loss;        /* HOST [n_microbatches] or NULL: loss of every micro-batch                */
  int32_t* delta;       /* HOST [S * n_microbatches] or NULL: Delta_{m,s} at [s*n + m]             */
  int64_t* version;     /* HOST [S] or NULL: local update index per stage after the run            */
  int32_t* max_q;       /* HOST [S] or NULL: largest unresolved-forward count seen per stage       */
  int64_t  n_slots;     /* out: logical slots the canonical schedule took                          */
  int64_t  n_launches;  /* out: kernels launched by the library during the run                     */
  float    elapsed_ms;  /* out: device time, first op to last op (CUDA events)                     */
} paci_run_report;

/* Bytes of DEVICE workspace for the inter-stage queues (activation / gradient rings, token staging). */
size_t paci_pipeline_workspace_bytes(paci_stage_t* const* stages, int32_t n_stages);
/* Creates one non-blocking stream per stage plus the ring events.  stages[s] must have stage_index s. */
int paci_pipeline_create(paci_stage_t* const* stages, int32_t n_stages, void* dev_ws, size_t ws_bytes,
                         paci_pipeline_t** out);
int paci_pipeline_destroy(paci_pipeline_t* p);
/* Run n_microbatches through the pipeline in the canonical logical schedule: per logical
 * slot every stage does at most one op, a message produced in slot tau is visible in slot tau+1,
 * backward before forward; the admission rule is enforced by paci_forward itself.
 *   tokens: int32 [n_microbatches, mu, T+1]; column t+1 is the target of column t.  n_microbatches = 0 is a no-op
 *           (tokens may be NULL): nothing is launched, no update happens, the report has 0 slots and launches.
 *           tokens_on_host = 0: DEVICE pointer.  1: HOST pointer (pinned or pageable); the run then
 *           includes the host->device copy of every micro-batch's tokens and the device->host read
 *           of its loss.
 *   mode PACI_MODE_FLUSH: micro-batches are grouped k at a time and no forward of group g+1 is
 *           issued at a stage before that stage applied update g.
 * Blocks until the run is complete. */
int paci_pipeline_run(paci_pipeline_t* p, const int32_t* tokens, int32_t tokens_on_host,
                      int64_t n_microbatches, int32_t mode, float lr, void* stream, paci_run_report* rep);
/* `stream` (both calls): the CALLER's stream.  The run is ordered after everything already enqueued on it (the
 * producer of a DEVICE token buffer, a non-blocking copy from pinned memory); NULL = the legacy default stream.
 * The stage streams are the pipeline's own.  Token ids are validated on the device: PACI_EINVAL after the run if
 * any id was outside [0, vocab) (the kernels clamp, so no access is out of bounds).
 *
 * paci_pipeline_run_var: heterogeneous micro-batch sizes.  n_seq: HOST int32 [n_microbatches], each in
 * [1, micro_batch] (NULL = all micro_batch); micro-batch m uses the first n_seq[m] sequences of tokens[m].
 * lr_by_update: HOST float [n_updates] or NULL: learning rate of a stage's u-th update DURING THIS RUN (u =
 * version - version at the start of the run), e.g. filled from paci_lr_schedule; NULL = constant lr. */
int paci_pipeline_run_var(paci_pipeline_t* p, const int32_t* tokens, int32_t tokens_on_host,
                          int64_t n_microbatches, const int32_t* n_seq, int32_t mode, float lr,
                          const float* lr_by_update, int64_t n_updates, void* stream, paci_run_report* rep);

/* ---- memory-constrained pipeline partitioning (App. D.5, Eq. 12-15; host arithmetic only) ---------- */
/* Splits n_layers sequential layers into n_stages contiguous groups minimising the slowest stage's time
 * max_j sum t_l subject to  sum s_l + w_j sum a_l <= budget  for every stage j, w_j = n_stages - j + 1 in-flight
 * micro-batches (Eq. 12-13; "the first stage carries N microbatches, the last carries one"), by the paper's
 * two-pass dynamic program (Eq. 15; infeasibility fallback: minimise the worst overshoot, ties by the maximum stage
 * time).
 *   t, s, a   HOST double [n_layers]: forward time, static bytes (parameters, gradients, optimizer state) and
 *             activation bytes per micro-batch of each layer (any consistent units)
 *   cuts      HOST int32 [n_stages + 1], out: 0 = c_0 < c_1 < ... < c_N = n_layers
 *   max_stage_time, max_overshoot   HOST, out (may be NULL)
 * Returns 0 (feasible: Eq. 13's optimum), 1 (budget infeasible: the fallback's partition), or PACI_EINVAL. */
int paci_partition(int32_t n_layers, int32_t n_stages, const double* t, const double* s, const double* a,
                   double budget, int32_t* cuts, double* max_stage_time, double* max_overshoot);

/* ---- op-level entry points (kernel parity tests and per-kernel roofline measurements) ------ */
/* All pointers DEVICE.  dtype = PACI_FP32 | PACI_BF16 selects the activation type T below. */

/* GEMM  C[M,N] (+)= op(A) op(B) (+ bias).  lda, ldb, ldc = row strides in elements.  layout:
 *   0 "NT" forward  : A[M,K] row-major, B[N,K] row-major (y = x W^T)         (SURVEY a3,a5,a7,a9,a10)
 *   1 "NN" dgrad    : A[M,K] row-major, B[K,N] row-major (dx = dy W)         (a13, current W: Eq. 1)
 *   2 "TN" wgrad    : A[K,M] row-major, B[K,N] row-major (dW = dy^T x)       (a14)
 * out_f32_accum = 0: C is T, overwritten, bias (fp32 [N], may be NULL) added.
 * out_f32_accum = 1: C is fp32 and the product is ADDED into it (beta = 1, Alg. 1 line 13).
 * PACI_BF16: all leading dimensions and pointers must be multiples of 8 elements / 16 bytes. */
int paci_op_gemm(int dtype, int layout, int M, int N, int K, const void* A, int lda, const void* B, int ldb,
                 const float* bias, void* C, int ldc, int out_f32_accum, void* stream);
/* The backward pair of one linear layer y = x W^T (rows a13 + a14): G_W[N_out, K_in] += dy^T x (fp32, beta = 1, Alg. 1
 * line 13) and dx[M, K_in] = dy W (the CURRENT W, Eq. 1).  dy [M, N_out], x [M, K_in], W [N_out, K_in], all row-major T
 * with the given row strides.  PACI_BF16: ONE tcgen05 launch -- the dgrad's tiles are dealt round-robin over the CTA
 * pairs and the wgrad's (tile, k-block) units are poured on top until every pair carries the same number of k-blocks. */
int paci_op_gemm_backward_pair(int dtype, int M, int N_out, int K_in, const void* dy, int ld_dy, const void* x, int ld_x,
                               const void* W, int ld_w, float* G_W, int ld_g, void* dx, int ld_dx, void* stream);
/* MLP-up with the activation fused (rows a7 + a8):  C = A B^T + bias (the pre-activation, which backward needs)
 * and G = gelu(C), both [M, N] of T with row stride ldc, A[M,K], B[N,K] row-major.  PACI_BF16 on the tcgen05 path:
 * ONE launch, gelu of the rounded C is computed in the GEMM epilogue and leaves through a second TMA store;
 * otherwise the GEMM followed by the GELU kernel (needs ldc == N). */
int paci_op_gemm_bias_gelu(int dtype, int M, int N, int K, const void* A, int lda, const void* B, int ldb,
                           const float* bias, void* C, void* G, int ldc, void* stream);
/* y = LN(x (+ res)) with gain g, bias b (fp32 [D]); writes xsum = x + res if xsum != NULL, and
 * mean, rstd (fp32 [rows]).  (a2, a6) */
int paci_op_layernorm_fwd(int dtype, int rows, int D, const void* x, const void* res, const float* g,
                          const float* b, void* xsum, void* y, float* mean, float* rstd, void* stream);
/* dx = (dres ? dres : 0) + LNbwd(dy; x, mean, rstd, g);  Gg += sum dy*xhat;  Gb += sum dy;
 * if Gcol != NULL: Gcol += column sums of dx.  (a18, a15) */
int paci_op_layernorm_bwd(int dtype, int rows, int D, const void* dy, const void* x, const float* mean,
                          const float* rstd, const float* g, const void* dres, void* dx, float* Gg,
                          float* Gb, float* Gcol, void* stream);
int paci_op_gelu_fwd(int dtype, size_t n, const void* p, void* out, void* stream);          /* a8  */
/* dp = dg * gelu'(p);  if Gbias != NULL: Gbias[cols] += column sums of dp.  (a16, a15) */
int paci_op_gelu_bwd(int dtype, int rows, int cols, const void* dg, const void* p, void* dp,
                     float* Gbias, void* stream);
/* G[cols] += column sums of x[rows, cols].  (a15) */
int paci_op_colsum(int dtype, int rows, int cols, const void* x, float* G, void* stream);
/* Causal attention over packed qkv [mu,T,3D] -> o [mu,T,D], lse fp32 [mu,H,T].  (a4) */
int paci_op_attention_fwd(int dtype, int mu, int T, int H, int dh, const void* qkv, void* o, float* lse,
                          void* stream);
/* dqkv [mu,T,3D] from do, qkv, o, lse; scratch: fp32 [mu*H*T] (+ [mu*T*D] fp32 in bf16 mode). (a17) */
int paci_op_attention_bwd(int dtype, int mu, int T, int H, int dh, const void* dout, const void* qkv,
                          const void* o, const float* lse, void* dqkv, float* scratch, void* stream);
size_t paci_op_attention_bwd_scratch_bytes(int dtype, int mu, int T, int H, int dh);
/* Backward of the attention output projection y = o Wo^T (rows a13 + a14 of that layer, and the prologue of a17):
 * G_Wo[D, D] += dy^T o (fp32) and d_o[mu T, D] = dy Wo, D = H dh, everything dense row-major (device pointers).
 * PACI_BF16 with dh = 64, T % 128 = 0 and lse, attn_scratch non-NULL: ONE tcgen05 launch whose dgrad epilogue also
 * writes, for every (b, h, t), delta = sum_d d_o[b,t,h,d] o[b,t,h,d] (the row term of softmax's backward, from the
 * ROUNDED d_o it stores) and lse log2(e) into attn_scratch (>= paci_op_attention_bwd_scratch_bytes, the layout
 * paci_op_attention_bwd uses); *prepared (host int) = 1, and paci_op_attention_bwd_prepared then runs without the
 * separate delta pass.  Any other case: the plain backward pair, *prepared = 0.  Errors: PACI_EINVAL (NULL prepared,
 * misaligned pointers), CUDA errors as everywhere. */
int paci_op_out_proj_backward(int dtype, int mu, int T, int H, int dh, const void* dy, const void* o, const void* Wo,
                              float* G_Wo, void* d_o, const float* lse, float* attn_scratch, int* prepared,
                              void* stream);
/* paci_op_attention_bwd for a scratch that paci_op_out_proj_backward prepared (*prepared = 1) on the same stream with
 * the same mu, T, H and the d_o passed here as dout.  PACI_BF16 only has such a path; other dtypes ignore the promise
 * and recompute. */
int paci_op_attention_bwd_prepared(int dtype, int mu, int T, int H, int dh, const void* dout, const void* qkv,
                                   const void* o, const float* lse, void* dqkv, float* scratch, void* stream);
/* paci_op_attention_bwd WITHOUT caller scratch and without any allocation, for callers that cannot call cudaMalloc
 * (CUDA graph capture, tight serving loops, harnesses that forbid it): same inputs, same outputs, same kernels; the
 * scratch is a file-scope `static __device__` array of PACI_ATTENTION_BWD_STATIC_MAX_BYTES inside the library, held by
 * every GPU that loads the library until the process exits.  All pointers are device pointers, layouts as in
 * paci_op_attention_bwd.  Limit: paci_op_attention_bwd_scratch_bytes(dtype, mu, T, H, dh) must not exceed the array
 * (bf16: 8 mu H T + 64 bytes, i.e. mu*H*T <= 524 312 -- configs[4]'s mu 8, H 20, T 1024 needs 1.3 MB); a larger shape
 * returns PACI_EINVAL with the sizes in paci_last_error() and launches nothing.  Every call on a device shares the
 * array and it keeps the last call's contents; each call rewrites what it reads (delta, lse*log2(e), the two work
 * counters) in stream order before reading it, so calls serialised on one stream or by events are independent, while
 * calls that OVERLAP on the GPU race and give wrong results: serialise them.  Calls no cudaMalloc / cudaFree.
 * (With paci_profile_begin active the sampling profiler creates events; do not profile inside a capture.) */
#define PACI_ATTENTION_BWD_STATIC_MAX_BYTES (4u * 1024u * 1024u + 256u)
int paci_op_attention_bwd_static(int dtype, int mu, int T, int H, int dh, const void* dout, const void* qkv,
                                 const void* o, const float* lse, void* dqkv, void* stream);
/* x = wte[tok] + wpe[pos] (a1);  tok int32 [mu,T]; wte [vocab, D], wpe fp32.  Ids outside [0, vocab) are clamped. */
int paci_op_embed_fwd(int dtype, int mu, int T, int D, int vocab, const int32_t* tok, const float* wte,
                      const float* wpe, void* x, void* stream);
/* Gwte[tok] += dx;  Gwpe[t] += sum_b dx  (a19). */
int paci_op_embed_bwd(int dtype, int mu, int T, int D, int vocab, const int32_t* tok, const void* dx, float* Gwte,
                      float* Gwpe, void* stream);
/* Dropout with the counter-based mask of paci_stage_config.dropout_seed: element e of x (n elements, T) is
 * kept iff word e % 4 of Philox4x32-10(counter = (e/4 lo, e/4 hi, (uint32) mb_id, site), key = (seed lo, seed hi))
 * is >= floor(p 2^32); kept values are multiplied by 1/(1-p).  out may alias x.  Forward and backward apply the
 * same map. */
int paci_op_dropout(int dtype, size_t n, const void* x, void* out, float p, uint64_t seed, int64_t mb_id,
                    int32_t site, void* stream);
/* loss[0] += sum_rows (lse - z[tgt]) / rows;  z <- dz = (softmax(z) - onehot) / rows in place.
 * z is [rows, ldz] with V valid columns (padding columns are written 0).  (a11) */
int paci_op_softmax_ce(int dtype, int rows, int V, int ldz, void* z, const int32_t* tgt, float* loss,
                       void* stream);
/* Fused AdamW over a flat arena of n fp32 elements, the first n_decay of which decay (a20):
 * g = G/k; w *= 1 - lr*wd (decayed part); m, v, bias-corrected update with step t; G = 0;
 * shadow (bf16, may be NULL) = bf16(w); *version_word += 1 (may be NULL). */
int paci_op_adamw(size_t n, size_t n_decay, float* w, float* m, float* v, float* G, void* shadow_bf16,
                  int k, int64_t t, float lr, float beta1, float beta2, float eps, float weight_decay,
                  int64_t* version_word, void* stream);

/* ---- sampled kernel timing (bench.py "roofline") ----------------------------- */
/* Categories, in order: gemm_fwd, gemm_dgrad, gemm_wgrad, attention_fwd, attention_bwd, layernorm_fwd,
 * layernorm_bwd, gelu_fwd, gelu_bwd, colsum, embedding, softmax_ce, adamw, other, gemm_bwd_pair.  flops / bytes are
 * the ALGORITHMIC work of the op, summed over every launch since
 * paci_profile_begin; every sample_stride-th launch is bracketed by CUDA events on the stream it is
 * launched on, and sampled_* sum those launches only (sampled_ms = their device time). */
#define PACI_PROF_NCAT 15
typedef struct paci_prof_entry {
  int64_t launches, sampled;
  double flops, bytes, sampled_flops, sampled_bytes, sampled_ms;
} paci_prof_entry;
int paci_profile_begin(int32_t sample_stride);      /* 0 switches the profiler off                */
int paci_profile_end(paci_prof_entry* out);         /* HOST [PACI_PROF_NCAT]; synchronises the device */
const char* paci_profile_category_name(int32_t cat);

/* Number of kernels the library has launched in this process (for bench.py's gpu_launches). */
int64_t paci_launch_count(void);
/* Work decomposition the LAST PACI_BF16 GEMM launched from this thread took (tests assert the path they
 * mean to cover): out6 = {cta_group, block_n, splits, range_mode, grid, tiles}.  HOST int32 [6]. */
void paci_gemm_last_plan(int32_t* out6);

#ifdef __cplusplus
}
#endif
#endif /* PACI_H_ */
