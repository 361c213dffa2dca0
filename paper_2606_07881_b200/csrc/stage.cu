// stage.cu -- the paci_stage object: Algorithm 1's per-stage state and the orchestration
// of one forward / backward / update of a GPT-2 pre-LN block stack.  Host code only; every step of
// the path runs in the kernels of this library.
//
// Device workspace layout (all offsets 256-byte aligned):
//   W   fp32 [P]   master parameters, laid out [decayed tensors | non-decayed tensors]
//   Mo  fp32 [P]   Adam first moment        Vo fp32 [P]  Adam second moment
//   G   fp32 [P]   gradient accumulator (raw sum over the window; Alg. 1 line 13)
//   Wb  bf16 [P]   weight shadow read by the tcgen05 GEMMs (PACI_BF16 only; refreshed by AdamW)
//   ctl            device version word, (vF, vB) stamps
//   stash          S-s slots ("the first stage carries N microbatches, the last carries one")
//   scratch        forward / backward temporaries
#include <cstring>
#include <deque>
#include <unordered_map>
#include <vector>

#include "common.cuh"

namespace paci {

struct TensorInfo {
  std::string name;
  size_t offset, numel;
  bool decay;
};

struct BlockStash {   // byte offsets inside a slot
  size_t x_in, y1, qkv, o, x1, y2, p, g, mean1, rstd1, mean2, rstd2, lse;
};

static constexpr int LOG_CAP = 4096;

}  // namespace paci

using namespace paci;

struct paci_stage {
  paci_stage_config cfg;
  int dtype, L, D, H, dh, T, mu, M, V, Vpad, S, s, k;
  size_t esz;
  std::vector<TensorInfo> tensors;
  std::unordered_map<std::string, int> index;
  size_t P, n_decay;
  // device
  char* ws;
  float *W, *Mo, *Vo, *G;
  bf16* Wb;
  int64_t* dev_version;
  int64_t* dev_stamps;     // [LOG_CAP][2]
  int n_slots;
  size_t slot_bytes;
  char* stash;
  std::vector<BlockStash> bs;
  size_t off_tok, off_xf_in, off_xf, off_meanf, off_rstdf, off_z;
  // scratch
  char *sc_proj, *sc_emb, *sc_dxa, *sc_dxb, *sc_dx1, *sc_dD, *sc_dD2, *sc_d4, *sc_dqkv;
  float* sc_attn;
  // host state (Alg. 1 lines 1-3 + P:66)
  int64_t version;
  int q, c;
  int64_t n_forwards;
  struct Unresolved { int64_t mb; int slot; int64_t vF; int log_idx; };
  std::deque<Unresolved> fifo;
  struct LogEntry { int64_t mb; int32_t delta; bool done; };
  std::vector<LogEntry> log;                       // ring, index = forward ordinal % LOG_CAP
  std::unordered_map<int64_t, int> log_of;         // mb_id -> ring index
};

namespace paci {

int stage_cfg_field(const ::paci_stage* st, int field) {
  return reinterpret_cast<const int32_t*>(&st->cfg)[field];
}

static size_t build_tensors(const paci_stage_config& c, std::vector<TensorInfo>* out, size_t* n_decay) {
  const size_t D = c.d_model;
  std::vector<TensorInfo> dec, non;
  auto add = [&](std::vector<TensorInfo>& v, const std::string& n, size_t numel, bool d) {
    v.push_back({n, 0, numel, d});
  };
  if (c.has_embedding) {
    add(non, "wte", (size_t)c.vocab * D, false);
    add(non, "wpe", (size_t)c.seq_len * D, false);
  }
  for (int l = 0; l < c.n_layers; ++l) {
    const std::string p = "h." + std::to_string(l) + ".";
    add(non, p + "ln1.g", D, false);  add(non, p + "ln1.b", D, false);
    add(dec, p + "attn.wqkv", 3 * D * D, true);  add(non, p + "attn.bqkv", 3 * D, false);
    add(dec, p + "attn.wo", D * D, true);        add(non, p + "attn.bo", D, false);
    add(non, p + "ln2.g", D, false);  add(non, p + "ln2.b", D, false);
    add(dec, p + "mlp.w1", 4 * D * D, true);     add(non, p + "mlp.b1", 4 * D, false);
    add(dec, p + "mlp.w2", 4 * D * D, true);     add(non, p + "mlp.b2", D, false);
  }
  if (c.has_head) {
    add(non, "lnf.g", D, false);  add(non, "lnf.b", D, false);
    if (!c.has_embedding) add(non, "head.w", (size_t)c.vocab * D, false);   // DESIGN.md R8: no decay
  }
  size_t off = 0;
  for (auto& t : dec) { t.offset = off; off += t.numel; }
  *n_decay = off;
  for (auto& t : non) { t.offset = off; off += t.numel; }
  if (out) { *out = dec; out->insert(out->end(), non.begin(), non.end()); }
  return off;
}

static int validate(const paci_stage_config* c) {
  if (!c) return fail(PACI_EINVAL, "null config");
  if (c->n_stages < 1 || c->stage_index < 0 || c->stage_index >= c->n_stages)
    return fail(PACI_EINVAL, "stage_index %d / n_stages %d", c->stage_index, c->n_stages);
  if (c->n_layers < 0 || c->d_model <= 0 || c->n_heads <= 0 || c->seq_len <= 0 || c->micro_batch <= 0 ||
      c->k_accum <= 0)
    return fail(PACI_EINVAL, "non-positive dimension");
  if (c->d_model % c->n_heads) return fail(PACI_EINVAL, "d_model %% n_heads != 0");
  const int dh = c->d_model / c->n_heads;
  if (c->dtype == PACI_BF16) {
    if (c->d_model % 64) return fail(PACI_EINVAL, "PACI_BF16 needs d_model %% 64 == 0");
    if (dh != 64) return fail(PACI_EINVAL, "PACI_BF16 needs head dim 64 (got %d)", dh);
    if (c->seq_len % 64) return fail(PACI_EINVAL, "PACI_BF16 needs seq_len %% 64 == 0");
  } else if (c->dtype == PACI_FP32) {
    if (c->d_model % 4 || dh > 128) return fail(PACI_EINVAL, "PACI_FP32 needs d_model %% 4 == 0, head dim <= 128");
  } else {
    return fail(PACI_EINVAL, "dtype %d", c->dtype);
  }
  if ((c->has_embedding || c->has_head) && c->vocab <= 0) return fail(PACI_EINVAL, "vocab");
  if (c->n_layers == 0 && !c->has_embedding && !c->has_head) return fail(PACI_EINVAL, "empty stage");
  return PACI_OK;
}

struct Layout {
  size_t P, n_decay, off_W, off_M, off_V, off_G, off_Wb, off_ctl, off_stash, slot_bytes, off_scratch, total;
  int n_slots, Vpad;
  std::vector<BlockStash> bs;
  size_t off_tok, off_xf_in, off_xf, off_meanf, off_rstdf, off_z;
  size_t sc_proj, sc_emb, sc_dxa, sc_dxb, sc_dx1, sc_dD, sc_dD2, sc_d4, sc_dqkv, sc_attn;
};

static Layout make_layout(const paci_stage_config& c) {
  Layout L;
  L.P = build_tensors(c, nullptr, &L.n_decay);
  const size_t e = c.dtype == PACI_BF16 ? 2 : 4;
  const size_t M = (size_t)c.micro_batch * c.seq_len, D = c.d_model;
  L.Vpad = (c.vocab + 63) / 64 * 64;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
  L.off_W = take(L.P * 4); L.off_M = take(L.P * 4); L.off_V = take(L.P * 4); L.off_G = take(L.P * 4);
  L.off_Wb = take(c.dtype == PACI_BF16 ? L.P * 2 : 0);
  L.off_ctl = take(8 + (size_t)LOG_CAP * 2 * 8);
  // one stash slot
  size_t so = 0;
  auto stake = [&](size_t bytes) { size_t o = so; so = align_up(so + bytes, 256); return o; };
  L.off_tok = stake(c.has_embedding ? M * 4 : 0);
  L.bs.resize(c.n_layers);
  for (int l = 0; l < c.n_layers; ++l) {
    BlockStash& b = L.bs[l];
    b.x_in = stake(M * D * e); b.y1 = stake(M * D * e); b.qkv = stake(M * 3 * D * e); b.o = stake(M * D * e);
    b.x1 = stake(M * D * e);   b.y2 = stake(M * D * e); b.p = stake(M * 4 * D * e);   b.g = stake(M * 4 * D * e);
    b.mean1 = stake(M * 4); b.rstd1 = stake(M * 4); b.mean2 = stake(M * 4); b.rstd2 = stake(M * 4);
    b.lse = stake((size_t)c.micro_batch * c.n_heads * c.seq_len * 4);
  }
  L.off_xf_in = stake(c.has_head ? M * D * e : 0);
  L.off_xf = stake(c.has_head ? M * D * e : 0);
  L.off_meanf = stake(c.has_head ? M * 4 : 0);
  L.off_rstdf = stake(c.has_head ? M * 4 : 0);
  L.off_z = stake(c.has_head ? M * (size_t)L.Vpad * e : 0);
  L.slot_bytes = so;
  L.n_slots = c.n_stages - c.stage_index;          // d_s + 1 (Eq. 9: q <= d_s before admission)
  L.off_stash = take(L.slot_bytes * L.n_slots);
  L.off_scratch = off;
  L.sc_proj = take(M * D * e); L.sc_emb = take(c.has_embedding ? M * D * e : 0);
  L.sc_dxa = take(M * D * e); L.sc_dxb = take(M * D * e); L.sc_dx1 = take(M * D * e);
  L.sc_dD = take(M * D * e);  L.sc_dD2 = take(M * D * e); L.sc_d4 = take(M * 4 * D * e);
  L.sc_dqkv = take(M * 3 * D * e);
  L.sc_attn = take(attention_bwd_scratch_bytes(c.dtype, c.micro_batch, c.seq_len, c.n_heads, D / c.n_heads));
  L.total = off;
  return L;
}

}  // namespace paci

extern "C" {

const char* paci_last_error(void) { return g_last_error.c_str(); }
int64_t paci_launch_count(void) { return g_launches.load(); }
int paci_gemm_backend_is_tcgen05(void) { return gemm_backend_tcgen05() ? 1 : 0; }

size_t paci_stage_workspace_bytes(const paci_stage_config* cfg) {
  if (validate(cfg) != PACI_OK) return 0;
  return make_layout(*cfg).total;
}

size_t paci_stage_param_count(const paci_stage_config* cfg) {
  if (validate(cfg) != PACI_OK) return 0;
  size_t nd;
  return build_tensors(*cfg, nullptr, &nd);
}

int paci_stage_create(const paci_stage_config* cfg, void* dev_ws, size_t ws_bytes, void* stream,
                      paci_stage_t** out) {
  int rc = validate(cfg);
  if (rc != PACI_OK) return rc;
  if (!dev_ws || !out) return fail(PACI_EINVAL, "null pointer");
  if ((uintptr_t)dev_ws % 256) return fail(PACI_EINVAL, "workspace must be 256-byte aligned");
  Layout L = make_layout(*cfg);
  if (ws_bytes < L.total) return fail(PACI_EINVAL, "workspace too small: %zu < %zu", ws_bytes, L.total);
  paci_stage* st = new paci_stage();
  st->cfg = *cfg;
  st->dtype = cfg->dtype; st->L = cfg->n_layers; st->D = cfg->d_model; st->H = cfg->n_heads;
  st->dh = st->D / st->H; st->T = cfg->seq_len; st->mu = cfg->micro_batch; st->M = st->mu * st->T;
  st->V = cfg->vocab; st->Vpad = L.Vpad; st->S = cfg->n_stages; st->s = cfg->stage_index; st->k = cfg->k_accum;
  st->esz = cfg->dtype == PACI_BF16 ? 2 : 4;
  st->P = build_tensors(*cfg, &st->tensors, &st->n_decay);
  for (size_t i = 0; i < st->tensors.size(); ++i) st->index[st->tensors[i].name] = (int)i;
  st->ws = (char*)dev_ws;
  st->W = (float*)(st->ws + L.off_W); st->Mo = (float*)(st->ws + L.off_M); st->Vo = (float*)(st->ws + L.off_V);
  st->G = (float*)(st->ws + L.off_G);
  st->Wb = cfg->dtype == PACI_BF16 ? (bf16*)(st->ws + L.off_Wb) : nullptr;
  st->dev_version = (int64_t*)(st->ws + L.off_ctl);
  st->dev_stamps = st->dev_version + 1;
  st->n_slots = L.n_slots; st->slot_bytes = L.slot_bytes; st->stash = st->ws + L.off_stash; st->bs = L.bs;
  st->off_tok = L.off_tok; st->off_xf_in = L.off_xf_in; st->off_xf = L.off_xf; st->off_meanf = L.off_meanf;
  st->off_rstdf = L.off_rstdf; st->off_z = L.off_z;
  st->sc_proj = st->ws + L.sc_proj; st->sc_emb = st->ws + L.sc_emb; st->sc_dxa = st->ws + L.sc_dxa;
  st->sc_dxb = st->ws + L.sc_dxb; st->sc_dx1 = st->ws + L.sc_dx1; st->sc_dD = st->ws + L.sc_dD;
  st->sc_dD2 = st->ws + L.sc_dD2; st->sc_d4 = st->ws + L.sc_d4; st->sc_dqkv = st->ws + L.sc_dqkv;
  st->sc_attn = (float*)(st->ws + L.sc_attn);
  st->version = 0; st->q = 0; st->c = 0; st->n_forwards = 0;
  st->log.assign(LOG_CAP, {-1, -1, false});
  cudaStream_t cs = (cudaStream_t)stream;
  cudaError_t e = cudaMemsetAsync(st->Mo, 0, (L.off_Wb - L.off_M), cs);          // m, v, G
  if (e == cudaSuccess) e = cudaMemsetAsync(st->dev_version, 0, 8 + (size_t)LOG_CAP * 16, cs);
  if (e != cudaSuccess) {
    delete st;
    return fail(PACI_ECUDA, "memset: %s", cudaGetErrorString(e));
  }
  *out = st;
  return PACI_OK;
}

int paci_stage_destroy(paci_stage_t* st) {
  delete st;
  return PACI_OK;
}

size_t paci_stage_tensor_numel(const paci_stage_t* st, const char* name) {
  if (!st || !name) return 0;
  auto it = st->index.find(name);
  return it == st->index.end() ? 0 : st->tensors[it->second].numel;
}

static float* group_ptr(paci_stage_t* st, int what) {
  switch (what) {
    case PACI_PARAM: return st->W;
    case PACI_GRAD_ACCUM: return st->G;
    case PACI_ADAM_M: return st->Mo;
    case PACI_ADAM_V: return st->Vo;
  }
  return nullptr;
}

int paci_stage_load(paci_stage_t* st, int what, const char* name, const float* host_src, size_t n, void* stream) {
  if (!st || !name || !host_src) return fail(PACI_EINVAL, "null pointer");
  auto it = st->index.find(name);
  if (it == st->index.end()) return fail(PACI_EINVAL, "no tensor '%s' on this stage", name);
  const TensorInfo& t = st->tensors[it->second];
  float* base = group_ptr(st, what);
  if (!base) return fail(PACI_EINVAL, "group %d", what);
  if (n != t.numel) return fail(PACI_EINVAL, "'%s' has %zu elements, got %zu", name, t.numel, n);
  cudaStream_t cs = (cudaStream_t)stream;
  PACI_CUDA_OK(cudaMemcpyAsync(base + t.offset, host_src, n * 4, cudaMemcpyHostToDevice, cs));
  if (what == PACI_PARAM && st->Wb) {
    int rc = cast_shadow(n, st->W + t.offset, st->Wb + t.offset, cs);
    if (rc) return rc;
  }
  PACI_CUDA_OK(cudaStreamSynchronize(cs));
  return PACI_OK;
}

int paci_stage_read(paci_stage_t* st, int what, const char* name, float* host_dst, size_t n, void* stream) {
  if (!st || !name || !host_dst) return fail(PACI_EINVAL, "null pointer");
  auto it = st->index.find(name);
  if (it == st->index.end()) return fail(PACI_EINVAL, "no tensor '%s' on this stage", name);
  const TensorInfo& t = st->tensors[it->second];
  float* base = group_ptr(st, what);
  if (!base) return fail(PACI_EINVAL, "group %d", what);
  if (n != t.numel) return fail(PACI_EINVAL, "'%s' has %zu elements, got %zu", name, t.numel, n);
  cudaStream_t cs = (cudaStream_t)stream;
  PACI_CUDA_OK(cudaMemcpyAsync(host_dst, base + t.offset, n * 4, cudaMemcpyDeviceToHost, cs));
  PACI_CUDA_OK(cudaStreamSynchronize(cs));
  return PACI_OK;
}

int64_t paci_version(const paci_stage_t* st) { return st ? st->version : -1; }
int32_t paci_unresolved(const paci_stage_t* st) { return st ? st->q : -1; }
int32_t paci_window_count(const paci_stage_t* st) { return st ? st->c : -1; }

int32_t paci_crossed_updates(const paci_stage_t* st, int64_t mb_id) {
  if (!st) return -1;
  auto it = st->log_of.find(mb_id);
  if (it == st->log_of.end()) return -1;
  const auto& e = st->log[it->second];
  return (e.mb == mb_id && e.done) ? e.delta : -1;
}

int paci_stage_device_stamps(paci_stage_t* st, int64_t mb_id, int64_t* vF, int64_t* vB, void* stream) {
  if (!st || !vF || !vB) return fail(PACI_EINVAL, "null pointer");
  auto it = st->log_of.find(mb_id);
  if (it == st->log_of.end() || st->log[it->second].mb != mb_id) return fail(PACI_EINVAL, "unknown mb_id");
  int64_t h[2];
  cudaStream_t cs = (cudaStream_t)stream;
  PACI_CUDA_OK(cudaMemcpyAsync(h, st->dev_stamps + 2 * (size_t)it->second, 16, cudaMemcpyDeviceToHost, cs));
  PACI_CUDA_OK(cudaStreamSynchronize(cs));
  *vF = h[0];
  *vB = h[1];
  return PACI_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
namespace paci {

struct Wref {   // pointers to one tensor in every group
  float* w; float* g; const void* wc;   // master, grad accumulator, compute-dtype weights (shadow or master)
};
static Wref wref(paci_stage* st, const std::string& name) {
  const TensorInfo& t = st->tensors[st->index.at(name)];
  Wref r;
  r.w = st->W + t.offset;
  r.g = st->G + t.offset;
  r.wc = st->Wb ? (const void*)(st->Wb + t.offset) : (const void*)(st->W + t.offset);
  return r;
}

#define RC(expr) do { int rc__ = (expr); if (rc__ != PACI_OK) return rc__; } while (0)

static int forward_impl(paci_stage* st, char* slot, const void* in, const int32_t* targets, void* out,
                        cudaStream_t cs) {
  const int dt = st->dtype, M = st->M, D = st->D;
  const void* xa;           // residual stream = xa (+ xb)
  const void* xb = nullptr;
  if (st->cfg.has_embedding) {
    int32_t* tok = (int32_t*)(slot + st->off_tok);
    PACI_CUDA_OK(cudaMemcpyAsync(tok, in, (size_t)M * 4, cudaMemcpyDeviceToDevice, cs));
    Wref wte = wref(st, "wte"), wpe = wref(st, "wpe");
    RC(embed_fwd(dt, st->mu, st->T, D, tok, wte.w, wpe.w, st->sc_emb, cs));
    xa = st->sc_emb;
  } else {
    xa = in;
  }
  for (int l = 0; l < st->L; ++l) {
    const BlockStash& b = st->bs[l];
    const std::string p = "h." + std::to_string(l) + ".";
    Wref ln1g = wref(st, p + "ln1.g"), ln1b = wref(st, p + "ln1.b"), wqkv = wref(st, p + "attn.wqkv"),
         bqkv = wref(st, p + "attn.bqkv"), wo = wref(st, p + "attn.wo"), bo = wref(st, p + "attn.bo"),
         ln2g = wref(st, p + "ln2.g"), ln2b = wref(st, p + "ln2.b"), w1 = wref(st, p + "mlp.w1"),
         b1 = wref(st, p + "mlp.b1"), w2 = wref(st, p + "mlp.w2"), b2 = wref(st, p + "mlp.b2");
    // a2: x_in = xa + xb (stashed), y1 = LN1(x_in)
    RC(ln_fwd(dt, M, D, xa, xb, ln1g.w, ln1b.w, slot + b.x_in, slot + b.y1, (float*)(slot + b.mean1),
              (float*)(slot + b.rstd1), cs));
    // a3: qkv = y1 Wqkv^T + b
    RC(gemm(dt, 0, M, 3 * D, D, slot + b.y1, D, wqkv.wc, D, bqkv.w, slot + b.qkv, 3 * D, 0, cs));
    // a4: causal attention
    RC(attention_fwd(dt, st->mu, st->T, st->H, st->dh, slot + b.qkv, slot + b.o, (float*)(slot + b.lse), cs));
    // a5: a = o Wo^T + b
    RC(gemm(dt, 0, M, D, D, slot + b.o, D, wo.wc, D, bo.w, st->sc_proj, D, 0, cs));
    // a6: x1 = x_in + a (stashed), y2 = LN2(x1)
    RC(ln_fwd(dt, M, D, slot + b.x_in, st->sc_proj, ln2g.w, ln2b.w, slot + b.x1, slot + b.y2,
              (float*)(slot + b.mean2), (float*)(slot + b.rstd2), cs));
    // a7: p = y2 W1^T + b1 ; a8: g = gelu(p)
    // gemm_bias_gelu (GELU in the GEMM epilogue) exists and is parity-clean, but with 4 epilogue warps its extra
    // epilogue work costs the MLP-up GEMM what the separate 4.7 TB/s kernel costs (measured: 0 net): not used yet.
    RC(gemm(dt, 0, M, 4 * D, D, slot + b.y2, D, w1.wc, D, b1.w, slot + b.p, 4 * D, 0, cs));
    RC(gelu_fwd(dt, (size_t)M * 4 * D, slot + b.p, slot + b.g, cs));
    // a9: m = g W2^T + b2 ; the residual add is fused into the next LayerNorm
    RC(gemm(dt, 0, M, D, 4 * D, slot + b.g, 4 * D, w2.wc, 4 * D, b2.w, st->sc_proj, D, 0, cs));
    xa = slot + b.x1;
    xb = st->sc_proj;
  }
  if (!st->cfg.has_head) return add_vec(dt, (size_t)M * D, xa, xb, out, cs);
  // a10: z = LN_f(x) Whead^T ; a11: loss and dz in place
  Wref lnfg = wref(st, "lnf.g"), lnfb = wref(st, "lnf.b");
  Wref head = wref(st, st->cfg.has_embedding ? "wte" : "head.w");
  RC(ln_fwd(dt, M, D, xa, xb, lnfg.w, lnfb.w, slot + st->off_xf_in, slot + st->off_xf,
            (float*)(slot + st->off_meanf), (float*)(slot + st->off_rstdf), cs));
  RC(gemm(dt, 0, M, st->V, D, slot + st->off_xf, D, head.wc, D, nullptr, slot + st->off_z, st->Vpad, 0, cs));
  PACI_CUDA_OK(cudaMemsetAsync(out, 0, sizeof(float), cs));
  return softmax_ce(dt, M, st->V, st->Vpad, slot + st->off_z, targets, (float*)out, cs);
}

static int backward_impl(paci_stage* st, char* slot, const void* dout, void* din, cudaStream_t cs) {
  const int dt = st->dtype, M = st->M, D = st->D;
  const void* dcur;                     // grad wrt the residual stream at the current depth
  float* pending_b2 = nullptr;          // G of the bias whose gradient is colsum(dcur)
  if (st->L > 0) pending_b2 = wref(st, "h." + std::to_string(st->L - 1) + ".mlp.b2").g;
  char* pp[2] = {st->sc_dxa, st->sc_dxb};
  int flip = 0;
  if (st->cfg.has_head) {
    Wref lnfg = wref(st, "lnf.g"), lnfb = wref(st, "lnf.b");
    Wref head = wref(st, st->cfg.has_embedding ? "wte" : "head.w");
    // a12: dxf = dz Whead (current weights, Eq. 1); G_head += dz^T xf (beta = 1 epilogue)
    RC(gemm(dt, 1, M, D, st->V, slot + st->off_z, st->Vpad, head.wc, D, nullptr, st->sc_dD, D, 0, cs));
    RC(gemm(dt, 2, st->V, D, M, slot + st->off_z, st->Vpad, slot + st->off_xf, D, nullptr, head.g, D, 1, cs));
    void* dst = (st->L == 0 && !st->cfg.has_embedding) ? din : (void*)pp[flip];
    RC(ln_bwd(dt, M, D, st->sc_dD, slot + st->off_xf_in, (float*)(slot + st->off_meanf),
              (float*)(slot + st->off_rstdf), lnfg.w, nullptr, dst, lnfg.g, lnfb.g, pending_b2, cs));
    pending_b2 = nullptr;
    dcur = dst;
    flip ^= 1;
  } else {
    dcur = dout;
  }
  for (int l = st->L - 1; l >= 0; --l) {
    const BlockStash& b = st->bs[l];
    const std::string p = "h." + std::to_string(l) + ".";
    Wref ln1g = wref(st, p + "ln1.g"), ln1b = wref(st, p + "ln1.b"), wqkv = wref(st, p + "attn.wqkv"),
         bqkv = wref(st, p + "attn.bqkv"), wo = wref(st, p + "attn.wo"), bo = wref(st, p + "attn.bo"),
         ln2g = wref(st, p + "ln2.g"), ln2b = wref(st, p + "ln2.b"), w1 = wref(st, p + "mlp.w1"),
         b1 = wref(st, p + "mlp.b1"), w2 = wref(st, p + "mlp.w2");
    if (pending_b2) {   // a15: only when dcur came from outside the stage (no producer to fuse into)
      RC(colsum(dt, M, D, dcur, pending_b2, cs));
      pending_b2 = nullptr;
    }
    // MLP-down: dg = dx2 W2 ; G_W2 += dx2^T g
    RC(gemm(dt, 1, M, 4 * D, D, dcur, D, w2.wc, 4 * D, nullptr, st->sc_d4, 4 * D, 0, cs));
    RC(gemm(dt, 2, D, 4 * D, M, dcur, D, slot + b.g, 4 * D, nullptr, w2.g, 4 * D, 1, cs));
    // a16: dp = dg * gelu'(p) in place ; G_b1 += colsum(dp)
    RC(gelu_bwd(dt, M, 4 * D, st->sc_d4, slot + b.p, st->sc_d4, b1.g, cs));
    // MLP-up: dy2 = dp W1 ; G_W1 += dp^T y2
    RC(gemm(dt, 1, M, D, 4 * D, st->sc_d4, 4 * D, w1.wc, D, nullptr, st->sc_dD, D, 0, cs));
    RC(gemm(dt, 2, 4 * D, D, M, st->sc_d4, 4 * D, slot + b.y2, D, nullptr, w1.g, D, 1, cs));
    // a18: dx1 = dx2 + LN2bwd(dy2) ; G_ln2 ; G_bo += colsum(dx1)
    RC(ln_bwd(dt, M, D, st->sc_dD, slot + b.x1, (float*)(slot + b.mean2), (float*)(slot + b.rstd2), ln2g.w, dcur,
              st->sc_dx1, ln2g.g, ln2b.g, bo.g, cs));
    // out-proj: do = dx1 Wo ; G_Wo += dx1^T o
    RC(gemm(dt, 1, M, D, D, st->sc_dx1, D, wo.wc, D, nullptr, st->sc_dD2, D, 0, cs));
    RC(gemm(dt, 2, D, D, M, st->sc_dx1, D, slot + b.o, D, nullptr, wo.g, D, 1, cs));
    // a17: attention backward
    RC(attention_bwd(dt, st->mu, st->T, st->H, st->dh, st->sc_dD2, slot + b.qkv, slot + b.o,
                     (float*)(slot + b.lse), st->sc_dqkv, st->sc_attn, bqkv.g, cs));   // + G_bqkv (a15)
    // QKV: dy1 = dqkv Wqkv ; G_Wqkv += dqkv^T y1
    RC(gemm(dt, 1, M, D, 3 * D, st->sc_dqkv, 3 * D, wqkv.wc, D, nullptr, st->sc_dD, D, 0, cs));
    RC(gemm(dt, 2, 3 * D, D, M, st->sc_dqkv, 3 * D, slot + b.y1, D, nullptr, wqkv.g, D, 1, cs));
    // a18: dx = dx1 + LN1bwd(dy1) ; G_ln1 ; colsum(dx) is the previous block's G_b2
    float* gcol = l > 0 ? wref(st, "h." + std::to_string(l - 1) + ".mlp.b2").g : nullptr;
    void* dst = (l == 0 && !st->cfg.has_embedding) ? din : (void*)pp[flip];
    RC(ln_bwd(dt, M, D, st->sc_dD, slot + b.x_in, (float*)(slot + b.mean1), (float*)(slot + b.rstd1), ln1g.w,
              st->sc_dx1, dst, ln1g.g, ln1b.g, gcol, cs));
    dcur = dst;
    flip ^= 1;
  }
  if (st->cfg.has_embedding) {
    Wref wte = wref(st, "wte"), wpe = wref(st, "wpe");
    // a19
    return embed_bwd(dt, st->mu, st->T, D, (const int32_t*)(slot + st->off_tok), dcur, wte.g, wpe.g, cs);
  }
  if (st->L == 0 && !st->cfg.has_head) return add_vec(dt, (size_t)M * D, dcur, nullptr, din, cs);
  return PACI_OK;
}

}  // namespace paci

extern "C" {

int paci_forward(paci_stage_t* st, int64_t mb_id, const void* in, const int32_t* targets, void* out,
                 void* stream) {
  if (!st || !in || !out) return fail(PACI_EINVAL, "null pointer");
  if (st->cfg.has_head && !targets) return fail(PACI_EINVAL, "head stage needs targets");
  if (st->c == st->k) return fail(PACI_ESTATE, "update pending: call paci_maybe_step first");
  for (const auto& u : st->fifo)
    if (u.mb == mb_id) return fail(PACI_ESTATE, "mb_id %lld is still unresolved", (long long)mb_id);
  // Alg. 1 line 5 / Eq. 9: admit iff q_s <= S-1-s
  if (st->q > st->S - 1 - st->s) return fail(PACI_EAGAIN, "admission: q=%d > d_s=%d", st->q, st->S - 1 - st->s);
  cudaStream_t cs = (cudaStream_t)stream;
  const int slot_i = (int)(st->n_forwards % st->n_slots);
  const int log_idx = (int)(st->n_forwards % LOG_CAP);
  char* slot = st->stash + (size_t)slot_i * st->slot_bytes;
  int rc = stamp_version(st->dev_version, st->dev_stamps + 2 * (size_t)log_idx, cs);
  if (rc == PACI_OK) rc = forward_impl(st, slot, in, targets, out, cs);
  if (rc != PACI_OK) return rc;
  // bookkeeping (Alg. 1 line 9): t^F = version, q += 1
  if (st->log[log_idx].mb >= 0) st->log_of.erase(st->log[log_idx].mb);
  st->log[log_idx] = {mb_id, -1, false};
  st->log_of[mb_id] = log_idx;
  st->fifo.push_back({mb_id, slot_i, st->version, log_idx});
  st->q += 1;
  st->n_forwards += 1;
  return PACI_OK;
}

int paci_backward(paci_stage_t* st, int64_t mb_id, const void* dout, void* din, void* stream) {
  if (!st) return fail(PACI_EINVAL, "null stage");
  if (st->cfg.has_head ? dout != nullptr : dout == nullptr)
    return fail(PACI_EINVAL, "dout must be NULL iff the stage has the head");
  if (st->cfg.has_embedding ? din != nullptr : din == nullptr)
    return fail(PACI_EINVAL, "din must be NULL iff the stage has the embedding");
  if (st->c == st->k) return fail(PACI_ESTATE, "update pending: call paci_maybe_step first");
  if (st->fifo.empty() || st->fifo.front().mb != mb_id)
    return fail(PACI_ESTATE, "backward of mb %lld is not the oldest unresolved forward", (long long)mb_id);
  const auto u = st->fifo.front();
  cudaStream_t cs = (cudaStream_t)stream;
  char* slot = st->stash + (size_t)u.slot * st->slot_bytes;
  int rc = stamp_version(st->dev_version, st->dev_stamps + 2 * (size_t)u.log_idx + 1, cs);
  if (rc == PACI_OK) rc = backward_impl(st, slot, dout, din, cs);
  if (rc != PACI_OK) return rc;
  // Eq. 8: Delta = t^B - t^F, read before line 16's test; lines 14-15: c += 1, q -= 1
  st->log[u.log_idx].delta = (int32_t)(st->version - u.vF);
  st->log[u.log_idx].done = true;
  st->fifo.pop_front();
  st->c += 1;
  st->q -= 1;
  return PACI_OK;
}

int paci_maybe_step(paci_stage_t* st, float lr, void* stream) {
  if (!st) return fail(PACI_EINVAL, "null stage");
  if (st->c != st->k) return 0;     // Alg. 1 line 16
  const paci_stage_config& c = st->cfg;
  int rc = adamw(st->P, st->n_decay, st->W, st->Mo, st->Vo, st->G, st->Wb, st->k, st->version + 1, lr, c.beta1,
                 c.beta2, c.eps, c.weight_decay, st->dev_version, (cudaStream_t)stream);
  if (rc != PACI_OK) return rc;
  st->version += 1;                 // lines 17-18
  st->c = 0;
  return 1;
}

}  // extern "C"
