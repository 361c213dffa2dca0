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
#include <cmath>
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

namespace paci {
struct Wref {   // pointers to one tensor in every group
  float* w; float* g; const void* wc;   // master, grad accumulator, compute-dtype weights (shadow or master)
};
struct BlockW { Wref ln1g, ln1b, wqkv, bqkv, wo, bo, ln2g, ln2b, w1, b1, w2, b2; };
}  // namespace paci

struct paci_stage {
  paci_stage_config cfg;
  int dtype, L, D, H, dh, T, mu, M, V, Vpad, S, s, k;
  size_t esz;
  std::vector<TensorInfo> tensors;
  std::unordered_map<std::string, int> index;
  std::vector<BlockW> bw;                          // per-block pointer table, built once at create
  Wref wte, wpe, lnfg, lnfb, head;
  size_t P, n_decay;
  // device
  char* ws;
  float *W, *Mo, *Vo, *G;
  bf16* Wb;
  int64_t* dev_version;
  int64_t* dev_err;        // sticky: a token / target id was out of range
  int64_t* dev_stamps;     // [LOG_CAP][2]
  int n_slots;
  size_t slot_bytes;       // of a stash slot: the full activation set, or (checkpoint) the stage input only
  char* stash;
  char* work_slot;         // checkpoint mode: the ONE full activation set, shared by forward and recompute
  size_t ck_in, ck_tgt;    // checkpoint mode: offsets of the stage input / targets inside a stash slot
  std::vector<BlockStash> bs;
  size_t off_tok, off_xf_in, off_xf, off_meanf, off_rstdf, off_z;
  // scratch
  char *sc_proj, *sc_emb, *sc_dxa, *sc_dxb, *sc_dx1, *sc_dD, *sc_dD2, *sc_d4, *sc_dqkv, *sc_dmask;
  float* sc_attn;
  float* sc_loss;
  // host state (Alg. 1 lines 1-3 + P:66)
  int64_t version;
  int q, c;
  int64_t n_forwards;
  struct Unresolved { int64_t mb; int slot; int64_t vF; int log_idx; int n_seq; };
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
    if (c->seq_len % 128) return fail(PACI_EINVAL, "PACI_BF16 needs seq_len %% 128 == 0");
  } else if (c->dtype == PACI_FP32) {
    if (c->d_model % 4 || dh > 128) return fail(PACI_EINVAL, "PACI_FP32 needs d_model %% 4 == 0, head dim <= 128");
  } else {
    return fail(PACI_EINVAL, "dtype %d", c->dtype);
  }
  if ((c->has_embedding || c->has_head) && c->vocab <= 0) return fail(PACI_EINVAL, "vocab");
  if (c->n_layers == 0 && !c->has_embedding && !c->has_head) return fail(PACI_EINVAL, "empty stage");
  if (c->checkpoint != 0 && c->checkpoint != 1) return fail(PACI_EINVAL, "checkpoint %d", c->checkpoint);
  if (!(c->dropout_p >= 0.f && c->dropout_p < 1.f)) return fail(PACI_EINVAL, "dropout_p %f", (double)c->dropout_p);
  return PACI_OK;
}

struct Layout {
  size_t P, n_decay, off_W, off_M, off_V, off_G, off_Wb, off_ctl, off_stash, slot_bytes, full_slot_bytes, off_scratch,
      total;
  int n_slots, Vpad;
  std::vector<BlockStash> bs;
  size_t off_tok, off_xf_in, off_xf, off_meanf, off_rstdf, off_z;
  size_t ck_in, ck_tgt, work_slot;
  size_t sc_proj, sc_emb, sc_dxa, sc_dxb, sc_dx1, sc_dD, sc_dD2, sc_d4, sc_dqkv, sc_attn, sc_dmask, sc_loss;
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
  L.off_ctl = take(16 + (size_t)LOG_CAP * 2 * 8);
  // one full activation set ("activations required for backpropagation", Alg. 1 line 7)
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
  L.full_slot_bytes = so;
  // checkpoint mode: a stash slot holds the stage input (and the targets) only
  size_t co = 0;
  auto ctake = [&](size_t bytes) { size_t o = co; co = align_up(co + bytes, 256); return o; };
  L.ck_in = ctake(c.has_embedding ? M * 4 : M * D * e);
  L.ck_tgt = ctake(c.has_head ? M * 4 : 0);
  L.slot_bytes = c.checkpoint ? co : so;
  L.n_slots = c.n_stages - c.stage_index;          // d_s + 1 (Eq. 9: q <= d_s before admission)
  L.off_stash = take(L.slot_bytes * L.n_slots);
  L.work_slot = take(c.checkpoint ? L.full_slot_bytes : 0);
  L.off_scratch = off;
  L.sc_proj = take(M * D * e); L.sc_emb = take(c.has_embedding ? M * D * e : 0);
  L.sc_dxa = take(M * D * e); L.sc_dxb = take(M * D * e); L.sc_dx1 = take(M * D * e);
  L.sc_dD = take(M * D * e);  L.sc_dD2 = take(M * D * e); L.sc_d4 = take(M * 4 * D * e);
  L.sc_dqkv = take(M * 3 * D * e);
  L.sc_attn = take(attention_bwd_scratch_bytes(c.dtype, c.micro_batch, c.seq_len, c.n_heads, D / c.n_heads));
  L.sc_dmask = take(c.dropout_p > 0.f ? M * D * e : 0);
  L.sc_loss = take(256);
  L.total = off;
  return L;
}

}  // namespace paci

extern "C" {

const char* paci_last_error(void) { return g_last_error.c_str(); }
int64_t paci_launch_count(void) { return g_launches.load(); }
void paci_gemm_last_plan(int32_t* out6) { if (out6) gemm_tc_last_plan(out6); }

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
  st->dev_err = st->dev_version + 1;
  st->dev_stamps = st->dev_version + 2;
  st->n_slots = L.n_slots; st->slot_bytes = L.slot_bytes; st->stash = st->ws + L.off_stash; st->bs = L.bs;
  st->work_slot = cfg->checkpoint ? st->ws + L.work_slot : nullptr;
  st->ck_in = L.ck_in; st->ck_tgt = L.ck_tgt;
  st->sc_dmask = cfg->dropout_p > 0.f ? st->ws + L.sc_dmask : nullptr;
  st->sc_loss = (float*)(st->ws + L.sc_loss);
  st->off_tok = L.off_tok; st->off_xf_in = L.off_xf_in; st->off_xf = L.off_xf; st->off_meanf = L.off_meanf;
  st->off_rstdf = L.off_rstdf; st->off_z = L.off_z;
  st->sc_proj = st->ws + L.sc_proj; st->sc_emb = st->ws + L.sc_emb; st->sc_dxa = st->ws + L.sc_dxa;
  st->sc_dxb = st->ws + L.sc_dxb; st->sc_dx1 = st->ws + L.sc_dx1; st->sc_dD = st->ws + L.sc_dD;
  st->sc_dD2 = st->ws + L.sc_dD2; st->sc_d4 = st->ws + L.sc_d4; st->sc_dqkv = st->ws + L.sc_dqkv;
  st->sc_attn = (float*)(st->ws + L.sc_attn);
  st->version = 0; st->q = 0; st->c = 0; st->n_forwards = 0;
  st->log.assign(LOG_CAP, {-1, -1, false});
  // pointer tables: no string building or hashing on the issuing thread after this point
  auto ref = [&](const std::string& name) {
    const TensorInfo& t = st->tensors[st->index.at(name)];
    Wref r;
    r.w = st->W + t.offset;
    r.g = st->G + t.offset;
    r.wc = st->Wb ? (const void*)(st->Wb + t.offset) : (const void*)(st->W + t.offset);
    return r;
  };
  st->bw.resize(st->L);
  for (int l = 0; l < st->L; ++l) {
    const std::string p = "h." + std::to_string(l) + ".";
    st->bw[l] = BlockW{ref(p + "ln1.g"), ref(p + "ln1.b"), ref(p + "attn.wqkv"), ref(p + "attn.bqkv"), ref(p + "attn.wo"),
                       ref(p + "attn.bo"), ref(p + "ln2.g"),  ref(p + "ln2.b"),  ref(p + "mlp.w1"),    ref(p + "mlp.b1"),
                       ref(p + "mlp.w2"),  ref(p + "mlp.b2")};
  }
  st->wte = st->wpe = st->lnfg = st->lnfb = st->head = Wref{nullptr, nullptr, nullptr};
  if (cfg->has_embedding) { st->wte = ref("wte"); st->wpe = ref("wpe"); }
  if (cfg->has_head) {
    st->lnfg = ref("lnf.g"); st->lnfb = ref("lnf.b");
    st->head = ref(cfg->has_embedding ? "wte" : "head.w");
  }
  cudaStream_t cs = (cudaStream_t)stream;
  cudaError_t e = cudaMemsetAsync(st->Mo, 0, (L.off_Wb - L.off_M), cs);          // m, v, G
  if (e == cudaSuccess) e = cudaMemsetAsync(st->dev_version, 0, 16 + (size_t)LOG_CAP * 16, cs);
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

#define RC(expr) do { int rc__ = (expr); if (rc__ != PACI_OK) return rc__; } while (0)

// dropout sites (R23): 0 = embedding output, 1 + 2l = attention branch of block l, 2 + 2l = its MLP branch
static inline int site_attn(int l) { return 1 + 2 * l; }
static inline int site_mlp(int l) { return 2 + 2 * l; }

// One forward of the stage over n_seq sequences into the activation set `act` (a stash slot, or the checkpoint
// mode's work slot).  x: int32 tokens [n_seq, T] (already inside the stash) if has_embedding, else h [n_seq, T, D].
// out: h [n_seq, T, D] (may be NULL: recomputation does not need it), or float loss[1] on the head stage.
static int forward_impl(paci_stage* st, char* act, const void* x, const int32_t* targets, void* out, int n_seq,
                        int64_t mb_id, cudaStream_t cs) {
  const int dt = st->dtype, M = n_seq * st->T, D = st->D;
  const float pd = st->cfg.dropout_p;
  const uint64_t seed = st->cfg.dropout_seed;
  const void* xa;           // residual stream = xa (+ xb)
  const void* xb = nullptr;
  if (st->cfg.has_embedding) {
    RC(embed_fwd(dt, n_seq, st->T, D, (const int32_t*)x, st->wte.w, st->wpe.w, st->sc_emb, st->V, st->dev_err, cs));
    if (pd > 0.f) RC(dropout(dt, (size_t)M * D, st->sc_emb, st->sc_emb, pd, seed, mb_id, 0, cs));
    xa = st->sc_emb;
  } else {
    xa = x;
  }
  for (int l = 0; l < st->L; ++l) {
    const BlockStash& b = st->bs[l];
    const BlockW& w = st->bw[l];
    // a2: x_in = xa + xb (stashed), y1 = LN1(x_in)
    RC(ln_fwd(dt, M, D, xa, xb, w.ln1g.w, w.ln1b.w, act + b.x_in, act + b.y1, (float*)(act + b.mean1),
              (float*)(act + b.rstd1), cs));
    // a3: qkv = y1 Wqkv^T + b
    RC(gemm(dt, 0, M, 3 * D, D, act + b.y1, D, w.wqkv.wc, D, w.bqkv.w, act + b.qkv, 3 * D, 0, cs));
    // a4: causal attention
    RC(attention_fwd(dt, n_seq, st->T, st->H, st->dh, act + b.qkv, act + b.o, (float*)(act + b.lse), cs));
    // a5: a = o Wo^T + b
    RC(gemm(dt, 0, M, D, D, act + b.o, D, w.wo.wc, D, w.bo.w, st->sc_proj, D, 0, cs));
    if (pd > 0.f) RC(dropout(dt, (size_t)M * D, st->sc_proj, st->sc_proj, pd, seed, mb_id, site_attn(l), cs));
    // a6: x1 = x_in + a (stashed), y2 = LN2(x1)
    RC(ln_fwd(dt, M, D, act + b.x_in, st->sc_proj, w.ln2g.w, w.ln2b.w, act + b.x1, act + b.y2,
              (float*)(act + b.mean2), (float*)(act + b.rstd2), cs));
    // a7 + a8: p = y2 W1^T + b1 (stashed: backward needs gelu'(p)) and g = gelu(p), one launch in bf16 mode (the
    // activation is computed in the GEMM epilogue and leaves through a second TMA store)
    RC(gemm_bias_gelu(dt, M, 4 * D, D, act + b.y2, D, w.w1.wc, D, w.b1.w, act + b.p, act + b.g, 4 * D, cs));
    // a recomputation (checkpointed backward: out == NULL) of a stage without the head stops here on its last block:
    // nothing that backward reads comes after g (the MLP-down output only feeds the stage's output)
    if (l == st->L - 1 && out == nullptr && !st->cfg.has_head) return PACI_OK;
    // a9: m = g W2^T + b2 ; the residual add is fused into the next LayerNorm
    RC(gemm(dt, 0, M, D, 4 * D, act + b.g, 4 * D, w.w2.wc, 4 * D, w.b2.w, st->sc_proj, D, 0, cs));
    if (pd > 0.f) RC(dropout(dt, (size_t)M * D, st->sc_proj, st->sc_proj, pd, seed, mb_id, site_mlp(l), cs));
    xa = act + b.x1;
    xb = st->sc_proj;
  }
  if (!st->cfg.has_head) return out != nullptr ? add_vec(dt, (size_t)M * D, xa, xb, out, cs) : PACI_OK;
  // a10: z = LN_f(x) Whead^T ; a11: loss (mean over THIS micro-batch's tokens, R22) and dz in place
  RC(ln_fwd(dt, M, D, xa, xb, st->lnfg.w, st->lnfb.w, act + st->off_xf_in, act + st->off_xf,
            (float*)(act + st->off_meanf), (float*)(act + st->off_rstdf), cs));
  RC(gemm(dt, 0, M, st->V, D, act + st->off_xf, D, st->head.wc, D, nullptr, act + st->off_z, st->Vpad, 0, cs));
  PACI_CUDA_OK(cudaMemsetAsync(out, 0, sizeof(float), cs));
  return softmax_ce(dt, M, st->V, st->Vpad, act + st->off_z, targets, (float*)out, st->dev_err, cs);
}

// Backward over the activation set `act` with the stage's CURRENT parameters (Eq. 1).  tok: the stashed
// int32 tokens (embedding stage).
static int backward_impl(paci_stage* st, char* act, const int32_t* tok, const void* dout, void* din, int n_seq,
                         int64_t mb_id, cudaStream_t cs) {
  const int dt = st->dtype, M = n_seq * st->T, D = st->D;
  const float pd = st->cfg.dropout_p;
  const uint64_t seed = st->cfg.dropout_seed;
  const bool drop = pd > 0.f;
  const void* dcur;                     // grad wrt the residual stream at the current depth
  // no dropout: colsum(dcur) IS the gradient of the last block's b2 and is fused into the producer of dcur (a15).
  // dropout: the branch gradient is mask o dcur / (1 - p), so the bias gradients are column sums of the masked copy.
  float* pending_b2 = (!drop && st->L > 0) ? st->bw[st->L - 1].b2.g : nullptr;
  char* pp[2] = {st->sc_dxa, st->sc_dxb};
  int flip = 0;
  if (st->cfg.has_head) {
    // a12: dxf = dz Whead (current weights, Eq. 1); G_head += dz^T xf (beta = 1 epilogue)
    RC(gemm(dt, 1, M, D, st->V, act + st->off_z, st->Vpad, st->head.wc, D, nullptr, st->sc_dD, D, 0, cs));
    RC(gemm(dt, 2, st->V, D, M, act + st->off_z, st->Vpad, act + st->off_xf, D, nullptr, st->head.g, D, 1, cs));
    void* dst = (st->L == 0 && !st->cfg.has_embedding) ? din : (void*)pp[flip];
    RC(ln_bwd(dt, M, D, st->sc_dD, act + st->off_xf_in, (float*)(act + st->off_meanf),
              (float*)(act + st->off_rstdf), st->lnfg.w, nullptr, dst, st->lnfg.g, st->lnfb.g, pending_b2, cs));
    pending_b2 = nullptr;
    dcur = dst;
    flip ^= 1;
  } else {
    dcur = dout;
  }
  for (int l = st->L - 1; l >= 0; --l) {
    const BlockStash& b = st->bs[l];
    const BlockW& w = st->bw[l];
    const void* dm = dcur;              // grad wrt the MLP branch output
    if (drop) {
      RC(dropout(dt, (size_t)M * D, dcur, st->sc_dmask, pd, seed, mb_id, site_mlp(l), cs));
      RC(colsum(dt, M, D, st->sc_dmask, w.b2.g, cs));
      dm = st->sc_dmask;
    } else if (pending_b2) {   // a15: only when dcur came from outside the stage (no producer to fuse into)
      RC(colsum(dt, M, D, dcur, pending_b2, cs));
      pending_b2 = nullptr;
    }
    // MLP-down: dg = dm W2 ; G_W2 += dm^T g   (a13 + a14: one launch for the pair)
    RC(gemm_backward_pair(dt, M, D, 4 * D, dm, D, act + b.g, 4 * D, w.w2.wc, 4 * D, w.w2.g, 4 * D, st->sc_d4, 4 * D, cs));
    // a16: dp = dg * gelu'(p) in place ; G_b1 += colsum(dp)
    RC(gelu_bwd(dt, M, 4 * D, st->sc_d4, act + b.p, st->sc_d4, w.b1.g, cs));
    // MLP-up: dy2 = dp W1 ; G_W1 += dp^T y2
    RC(gemm_backward_pair(dt, M, 4 * D, D, st->sc_d4, 4 * D, act + b.y2, D, w.w1.wc, D, w.w1.g, D, st->sc_dD, D, cs));
    // a18: dx1 = dcur + LN2bwd(dy2) ; G_ln2 ; G_bo += colsum(dx1) (no dropout)
    RC(ln_bwd(dt, M, D, st->sc_dD, act + b.x1, (float*)(act + b.mean2), (float*)(act + b.rstd2), w.ln2g.w, dcur,
              st->sc_dx1, w.ln2g.g, w.ln2b.g, drop ? nullptr : w.bo.g, cs));
    const void* da = st->sc_dx1;        // grad wrt the attention branch output
    if (drop) {
      RC(dropout(dt, (size_t)M * D, st->sc_dx1, st->sc_dmask, pd, seed, mb_id, site_attn(l), cs));
      RC(colsum(dt, M, D, st->sc_dmask, w.bo.g, cs));
      da = st->sc_dmask;
    }
    // out-proj: do = da Wo ; G_Wo += da^T o
    // (tcgen05 path: the dgrad's epilogue also leaves a17's delta = rowsum(do * o) and lse log2(e) in sc_attn)
    int attn_prepared = 0;
    RC(out_proj_backward(dt, n_seq, st->T, st->H, st->dh, da, act + b.o, w.wo.wc, w.wo.g, st->sc_dD2,
                         (float*)(act + b.lse), st->sc_attn, &attn_prepared, cs));
    // a17: attention backward
    RC(attention_bwd(dt, n_seq, st->T, st->H, st->dh, st->sc_dD2, act + b.qkv, act + b.o,
                     (float*)(act + b.lse), st->sc_dqkv, st->sc_attn, w.bqkv.g, cs, attn_prepared));   // + G_bqkv (a15)
    // QKV: dy1 = dqkv Wqkv ; G_Wqkv += dqkv^T y1
    RC(gemm_backward_pair(dt, M, 3 * D, D, st->sc_dqkv, 3 * D, act + b.y1, D, w.wqkv.wc, D, w.wqkv.g, D, st->sc_dD, D, cs));
    // a18: dx = dx1 + LN1bwd(dy1) ; G_ln1 ; colsum(dx) is the previous block's G_b2 (no dropout)
    float* gcol = (!drop && l > 0) ? st->bw[l - 1].b2.g : nullptr;
    void* dst = (l == 0 && !st->cfg.has_embedding) ? din : (void*)pp[flip];
    RC(ln_bwd(dt, M, D, st->sc_dD, act + b.x_in, (float*)(act + b.mean1), (float*)(act + b.rstd1), w.ln1g.w,
              st->sc_dx1, dst, w.ln1g.g, w.ln1b.g, gcol, cs));
    dcur = dst;
    flip ^= 1;
  }
  if (st->cfg.has_embedding) {
    if (drop) {
      RC(dropout(dt, (size_t)M * D, dcur, st->sc_dmask, pd, seed, mb_id, 0, cs));
      dcur = st->sc_dmask;
    }
    // a19
    return embed_bwd(dt, n_seq, st->T, D, tok, dcur, st->wte.g, st->wpe.g, st->V, cs);
  }
  if (st->L == 0 && !st->cfg.has_head) return add_vec(dt, (size_t)M * D, dcur, nullptr, din, cs);
  return PACI_OK;
}

}  // namespace paci

extern "C" {

int paci_forward_var(paci_stage_t* st, int64_t mb_id, int32_t n_seq, const void* in, const int32_t* targets,
                     void* out, void* stream) {
  if (!st || !in || !out) return fail(PACI_EINVAL, "null pointer");
  if (n_seq < 1 || n_seq > st->mu) return fail(PACI_EINVAL, "n_seq %d outside [1, micro_batch = %d]", n_seq, st->mu);
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
  const bool ck = st->cfg.checkpoint != 0;
  const size_t M = (size_t)n_seq * st->T;
  int rc = stamp_version(st->dev_version, st->dev_stamps + 2 * (size_t)log_idx, cs);
  if (rc != PACI_OK) return rc;
  // what backward needs of the stage INPUT goes into the stash: the tokens (embedding scatter-add), and in
  // checkpoint mode the whole input and the targets (the recomputation starts from them)
  const void* x = in;
  if (st->cfg.has_embedding) {
    int32_t* tok = (int32_t*)(slot + (ck ? st->ck_in : st->off_tok));
    PACI_CUDA_OK(cudaMemcpyAsync(tok, in, M * 4, cudaMemcpyDeviceToDevice, cs));
    x = tok;
  } else if (ck) {
    PACI_CUDA_OK(cudaMemcpyAsync(slot + st->ck_in, in, M * st->D * st->esz, cudaMemcpyDeviceToDevice, cs));
  }
  if (ck && st->cfg.has_head)
    PACI_CUDA_OK(cudaMemcpyAsync(slot + st->ck_tgt, targets, M * 4, cudaMemcpyDeviceToDevice, cs));
  rc = forward_impl(st, ck ? st->work_slot : slot, x, targets, out, n_seq, mb_id, cs);
  if (rc != PACI_OK) return rc;
  // bookkeeping (Alg. 1 line 9): t^F = version, q += 1
  const int64_t old = st->log[log_idx].mb;
  auto it = st->log_of.find(old);
  if (it != st->log_of.end() && it->second == log_idx) st->log_of.erase(it);   // only if it still maps to THIS entry
  st->log[log_idx] = {mb_id, -1, false};
  st->log_of[mb_id] = log_idx;
  st->fifo.push_back({mb_id, slot_i, st->version, log_idx, n_seq});
  st->q += 1;
  st->n_forwards += 1;
  return PACI_OK;
}

int paci_forward(paci_stage_t* st, int64_t mb_id, const void* in, const int32_t* targets, void* out,
                 void* stream) {
  if (!st) return fail(PACI_EINVAL, "null pointer");
  return paci_forward_var(st, mb_id, st->mu, in, targets, out, stream);
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
  if (rc != PACI_OK) return rc;
  if (st->cfg.checkpoint) {
    // "those activations are instead recomputed under the current parameter version before differentiation"
    const void* x = slot + st->ck_in;
    rc = forward_impl(st, st->work_slot, x, (const int32_t*)(slot + st->ck_tgt), st->cfg.has_head ? st->sc_loss : nullptr,
                      u.n_seq, mb_id, cs);
    if (rc == PACI_OK)
      rc = backward_impl(st, st->work_slot, (const int32_t*)x, dout, din, u.n_seq, mb_id, cs);
  } else {
    rc = backward_impl(st, slot, (const int32_t*)(slot + st->off_tok), dout, din, u.n_seq, mb_id, cs);
  }
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

int paci_stage_set_state(paci_stage_t* st, int64_t version, int32_t window_count, void* stream) {
  if (!st) return fail(PACI_EINVAL, "null stage");
  if (version < 0 || window_count < 0 || window_count >= st->k)
    return fail(PACI_EINVAL, "set_state: version %lld, window_count %d (k = %d)", (long long)version, window_count, st->k);
  if (st->q != 0) return fail(PACI_ESTATE, "set_state with %d unresolved forwards", st->q);
  cudaStream_t cs = (cudaStream_t)stream;
  PACI_CUDA_OK(cudaMemcpyAsync(st->dev_version, &version, 8, cudaMemcpyHostToDevice, cs));
  PACI_CUDA_OK(cudaStreamSynchronize(cs));
  st->version = version;
  st->c = window_count;
  return PACI_OK;
}

int paci_stage_check(paci_stage_t* st, void* stream) {
  if (!st) return fail(PACI_EINVAL, "null stage");
  cudaStream_t cs = (cudaStream_t)stream;
  int64_t e = 0;
  PACI_CUDA_OK(cudaMemcpyAsync(&e, st->dev_err, 8, cudaMemcpyDeviceToHost, cs));
  PACI_CUDA_OK(cudaStreamSynchronize(cs));
  if (e == 0) return PACI_OK;
  PACI_CUDA_OK(cudaMemsetAsync(st->dev_err, 0, 8, cs));
  PACI_CUDA_OK(cudaStreamSynchronize(cs));
  return fail(PACI_EINVAL, "stage %d: a token or target id was outside [0, %d) (clamped on the device)", st->s, st->V);
}

float paci_lr_schedule(int64_t step, int64_t total_steps, int64_t warmup_steps, float peak, float final_frac) {
  if (warmup_steps > 0 && step < warmup_steps) return peak * (float)((double)(step + 1) / (double)warmup_steps);
  if (step >= total_steps || total_steps <= warmup_steps) return peak * final_frac;
  const double prog = (double)(step - warmup_steps) / (double)(total_steps - warmup_steps);
  return (float)((double)peak * ((double)final_frac + (1.0 - (double)final_frac) * 0.5 * (1.0 + std::cos(3.14159265358979323846 * prog))));
}

}  // extern "C"
