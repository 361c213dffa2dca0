// pipeline.cu -- schedule driver: the S stages of the asynchronous 1F1B pipeline emulated on ONE GPU
// (BASELINE.json item 6).  Each stage has its own stream; the messages of Alg. 1
// lines 8 and 14 (h_{m,i} forward, grad h_{m,i-1} backward) travel through device-memory rings
// guarded by CUDA events.  Host code only.
//
// Logical schedule: time advances in slots; in a slot every
// stage does at most one op, decided from what was visible at the START of the slot (a message
// produced in slot tau is visible in slot tau+1); a ready backward goes before a ready forward (R1);
// the admission rule q <= S-1-s is enforced by paci_forward itself (PACI_EAGAIN -> the stage idles).
// This is an independent restatement of Alg. 1 -- it shares no code with oracle/schedule.py, and the
// crossed-update counts of the two must agree exactly.
#include <vector>

#include "common.cuh"

using namespace paci;

#define paci_stage_cfg_field ::paci::stage_cfg_field   // int32 field i of paci_stage_config (stage.cu)

namespace {
constexpr int RING = 2;           // messages per boundary and direction
constexpr int MAX_MB = 1 << 16;   // loss slots
}  // namespace

struct paci_pipeline {
  int S, mu, T, D, dtype, k;
  size_t esz, msg_bytes;
  std::vector<paci_stage_t*> st;
  std::vector<cudaStream_t> streams;
  cudaStream_t main;
  std::vector<char*> fbuf, bbuf;                       // [(S-1)*RING]
  std::vector<cudaEvent_t> f_ready, f_free, b_ready, b_free;
  int tok_ring;
  int32_t *tok_stage, *tok_in, *tok_tgt;               // [tok_ring][mu*(T+1)], [tok_ring][M], [tok_ring][M]
  float* loss;                                         // [MAX_MB]
  cudaEvent_t ev_start, ev_stop, ev_in;
  std::vector<cudaEvent_t> ev_done;
};

static size_t pipeline_layout(const paci_pipeline& p, std::vector<size_t>* offs) {
  size_t off = 0;
  auto take = [&](size_t b) { size_t o = off; off = align_up(off + b, 256); if (offs) offs->push_back(o); return o; };
  for (int i = 0; i < (p.S - 1) * RING * 2; ++i) take(p.msg_bytes);
  take((size_t)p.tok_ring * p.mu * (p.T + 1) * 4);
  take((size_t)p.tok_ring * p.mu * p.T * 4);
  take((size_t)p.tok_ring * p.mu * p.T * 4);
  take((size_t)MAX_MB * 4);
  return off;
}

static int fill_dims(paci_pipeline& p, paci_stage_t* const* stages, int32_t S) {
  if (!stages || S < 1) return fail(PACI_EINVAL, "pipeline: no stages");
  p.S = S;
  for (int s = 0; s < S; ++s) {
    if (!stages[s]) return fail(PACI_EINVAL, "pipeline: null stage %d", s);
    if (paci_stage_cfg_field(stages[s], 0) != s || paci_stage_cfg_field(stages[s], 1) != S)
      return fail(PACI_EINVAL, "pipeline: stage %d has stage_index %d / n_stages %d", s,
                  paci_stage_cfg_field(stages[s], 0), paci_stage_cfg_field(stages[s], 1));
  }
  p.D = paci_stage_cfg_field(stages[0], 3);
  p.T = paci_stage_cfg_field(stages[0], 5);
  p.mu = paci_stage_cfg_field(stages[0], 6);
  p.k = paci_stage_cfg_field(stages[0], 7);
  p.dtype = paci_stage_cfg_field(stages[0], 11);
  for (int s = 0; s < S; ++s) {
    if (paci_stage_cfg_field(stages[s], 3) != p.D || paci_stage_cfg_field(stages[s], 5) != p.T ||
        paci_stage_cfg_field(stages[s], 6) != p.mu || paci_stage_cfg_field(stages[s], 7) != p.k ||
        paci_stage_cfg_field(stages[s], 11) != p.dtype)
      return fail(PACI_EINVAL, "pipeline: stage %d disagrees on D/T/mu/k/dtype", s);
    if ((paci_stage_cfg_field(stages[s], 9) != 0) != (s == 0) ||
        (paci_stage_cfg_field(stages[s], 10) != 0) != (s == S - 1))
      return fail(PACI_EINVAL, "pipeline: embedding must be on stage 0 and the head on stage S-1");
  }
  p.esz = p.dtype == PACI_BF16 ? 2 : 4;
  p.msg_bytes = (size_t)p.mu * p.T * p.D * p.esz;
  p.tok_ring = S + 1;
  return PACI_OK;
}

extern "C" {

size_t paci_pipeline_workspace_bytes(paci_stage_t* const* stages, int32_t n_stages) {
  paci_pipeline p;
  if (fill_dims(p, stages, n_stages) != PACI_OK) return 0;
  return pipeline_layout(p, nullptr);
}

int paci_pipeline_create(paci_stage_t* const* stages, int32_t n_stages, void* dev_ws, size_t ws_bytes,
                         paci_pipeline_t** out) {
  if (!out || !dev_ws) return fail(PACI_EINVAL, "null pointer");
  paci_pipeline* p = new paci_pipeline();
  int rc = fill_dims(*p, stages, n_stages);
  if (rc != PACI_OK) { delete p; return rc; }
  std::vector<size_t> offs;
  const size_t need = pipeline_layout(*p, &offs);
  if (ws_bytes < need || (uintptr_t)dev_ws % 256) {
    delete p;
    return fail(PACI_EINVAL, "pipeline workspace: need %zu bytes, 256-byte aligned", need);
  }
  char* base = (char*)dev_ws;
  const int S = p->S, nb = (S - 1) * RING;
  p->st.assign(stages, stages + S);
  for (int i = 0; i < nb; ++i) p->fbuf.push_back(base + offs[i]);
  for (int i = 0; i < nb; ++i) p->bbuf.push_back(base + offs[nb + i]);
  p->tok_stage = (int32_t*)(base + offs[2 * nb]);
  p->tok_in = (int32_t*)(base + offs[2 * nb + 1]);
  p->tok_tgt = (int32_t*)(base + offs[2 * nb + 2]);
  p->loss = (float*)(base + offs[2 * nb + 3]);
  p->streams.resize(S);
  for (int s = 0; s < S; ++s) PACI_CUDA_OK(cudaStreamCreateWithFlags(&p->streams[s], cudaStreamNonBlocking));
  PACI_CUDA_OK(cudaStreamCreateWithFlags(&p->main, cudaStreamNonBlocking));
  auto mk = [&](std::vector<cudaEvent_t>& v, int n) -> int {
    v.resize(n);
    for (int i = 0; i < n; ++i) PACI_CUDA_OK(cudaEventCreateWithFlags(&v[i], cudaEventDisableTiming));
    return PACI_OK;
  };
  if ((rc = mk(p->f_ready, nb)) || (rc = mk(p->f_free, nb)) || (rc = mk(p->b_ready, nb)) ||
      (rc = mk(p->b_free, nb)) || (rc = mk(p->ev_done, S)))
    return rc;
  PACI_CUDA_OK(cudaEventCreate(&p->ev_start));
  PACI_CUDA_OK(cudaEventCreate(&p->ev_stop));
  PACI_CUDA_OK(cudaEventCreateWithFlags(&p->ev_in, cudaEventDisableTiming));
  *out = p;
  return PACI_OK;
}

int paci_pipeline_destroy(paci_pipeline_t* p) {
  if (!p) return PACI_OK;
  for (auto s : p->streams) cudaStreamDestroy(s);
  cudaStreamDestroy(p->main);
  for (auto* v : {&p->f_ready, &p->f_free, &p->b_ready, &p->b_free, &p->ev_done})
    for (auto e : *v) cudaEventDestroy(e);
  cudaEventDestroy(p->ev_start);
  cudaEventDestroy(p->ev_stop);
  cudaEventDestroy(p->ev_in);
  delete p;
  return PACI_OK;
}

int paci_pipeline_run(paci_pipeline_t* p, const int32_t* tokens, int32_t tokens_on_host, int64_t n,
                      int32_t mode, float lr, void* stream, paci_run_report* rep) {
  return paci_pipeline_run_var(p, tokens, tokens_on_host, n, nullptr, mode, lr, nullptr, 0, stream, rep);
}

int paci_pipeline_run_var(paci_pipeline_t* p, const int32_t* tokens, int32_t tokens_on_host, int64_t n,
                          const int32_t* n_seq, int32_t mode, float lr, const float* lr_by_update,
                          int64_t n_updates, void* stream, paci_run_report* rep) {
  if (!p || !rep || (!tokens && n > 0)) return fail(PACI_EINVAL, "null pointer");   // n = 0: tokens may be NULL
  if (n < 0 || n > MAX_MB) return fail(PACI_EINVAL, "n_microbatches %lld out of range", (long long)n);
  if (mode != PACI_MODE_PACI && mode != PACI_MODE_FLUSH) return fail(PACI_EINVAL, "mode %d", mode);
  if (n_seq)
    for (int64_t m = 0; m < n; ++m)
      if (n_seq[m] < 1 || n_seq[m] > p->mu)
        return fail(PACI_EINVAL, "n_seq[%lld] = %d outside [1, %d]", (long long)m, n_seq[m], p->mu);
  const int S = p->S, M = p->mu * p->T;
  const size_t tok_per_mb = (size_t)p->mu * (p->T + 1);
  for (int s = 0; s < S; ++s)
    if (paci_unresolved(p->st[s]) != 0 || paci_window_count(p->st[s]) != 0)
      return fail(PACI_ESTATE, "pipeline_run: stage %d is mid-window", s);
  std::vector<int64_t> v0(S);
  for (int s = 0; s < S; ++s) v0[s] = paci_version(p->st[s]);
  const int64_t launches0 = paci_launch_count();

  struct PeerGuard {   // sampled launches of the in-library profiler run exclusively w.r.t. the stage streams
    explicit PeerGuard(const std::vector<cudaStream_t>& v) { prof_set_peer_streams(v.data(), (int)v.size()); }
    ~PeerGuard() { prof_set_peer_streams(nullptr, 0); }
  } peer_guard(p->streams);
  // the run is ordered after everything already enqueued on the caller's stream (e.g. the producer of a device
  // token buffer); all stage streams start after ev_start
  PACI_CUDA_OK(cudaEventRecord(p->ev_in, (cudaStream_t)stream));
  PACI_CUDA_OK(cudaStreamWaitEvent(p->main, p->ev_in, 0));
  PACI_CUDA_OK(cudaEventRecord(p->ev_start, p->main));
  for (int s = 0; s < S; ++s) PACI_CUDA_OK(cudaStreamWaitEvent(p->streams[s], p->ev_start, 0));

  std::vector<int64_t> nf(S, 0), nb(S, 0), vis_f(S, 0), vis_b(S, 0), new_f(S, 0), new_b(S, 0);
  std::vector<int> max_q(S, 0);
  vis_f[0] = n;
  int64_t slots = 0;
  auto all_done = [&]() { for (int s = 0; s < S; ++s) if (nb[s] < n) return false; return true; };
  while (!all_done()) {
    bool progressed = false;
    for (int s = 0; s < S; ++s) {
      cudaStream_t cs = p->streams[s];
      const bool b_ready = nb[s] < nf[s] && vis_b[s] > nb[s];
      bool f_ready = nf[s] < n && vis_f[s] > nf[s];
      if (f_ready && mode == PACI_MODE_FLUSH)
        f_ready = nf[s] / p->k == paci_version(p->st[s]) - v0[s];   // group g+1 waits for update g
      if (b_ready) {
        const int64_t m = nb[s];
        const int r = (int)(m % RING);
        const void* dout = nullptr;
        void* din = nullptr;
        if (s < S - 1) {
          PACI_CUDA_OK(cudaStreamWaitEvent(cs, p->b_ready[s * RING + r], 0));
          dout = p->bbuf[s * RING + r];
        }
        if (s > 0) {
          if (m >= RING) {
            if (nb[s - 1] <= m - RING) continue;   // ring full: upstream has not consumed yet (never in canon)
            PACI_CUDA_OK(cudaStreamWaitEvent(cs, p->b_free[(s - 1) * RING + r], 0));
          }
          din = p->bbuf[(s - 1) * RING + r];
        }
        int rc = paci_backward(p->st[s], m, dout, din, cs);
        if (rc != PACI_OK) return rc;
        if (s < S - 1) PACI_CUDA_OK(cudaEventRecord(p->b_free[s * RING + r], cs));
        if (s > 0) PACI_CUDA_OK(cudaEventRecord(p->b_ready[(s - 1) * RING + r], cs));
        if (rep->delta) rep->delta[(size_t)s * n + m] = paci_crossed_updates(p->st[s], m);
        float lr_now = lr;                                   // LR schedule: indexed by the stage's own update count
        if (lr_by_update) {
          const int64_t u = paci_version(p->st[s]) - v0[s];
          if (paci_window_count(p->st[s]) == p->k && u >= n_updates)
            return fail(PACI_EINVAL, "pipeline_run: lr_by_update has %lld entries, update %lld needed", (long long)n_updates, (long long)u);
          if (u < n_updates) lr_now = lr_by_update[u];
        }
        rc = paci_maybe_step(p->st[s], lr_now, cs);
        if (rc < 0) return rc;
        nb[s] += 1;
        if (s > 0) new_b[s - 1] += 1;
        progressed = true;
      } else if (f_ready) {
        const int64_t m = nf[s];
        const int r = (int)(m % RING);
        if (s < S - 1 && m >= RING && nf[s + 1] <= m - RING) continue;   // ring full (never in canon)
        // admission is the stage's own decision (Alg. 1 line 5): probe before touching the streams
        if (paci_unresolved(p->st[s]) > S - 1 - s) continue;
        const void* in;
        const int32_t* tgt = nullptr;
        void* outp;
        const int tr = (int)(m % p->tok_ring);
        if (s == 0) {
          const int32_t* src = tokens + (size_t)m * tok_per_mb;
          if (tokens_on_host) {
            int32_t* stg = p->tok_stage + (size_t)tr * tok_per_mb;
            PACI_CUDA_OK(cudaMemcpyAsync(stg, src, tok_per_mb * 4, cudaMemcpyHostToDevice, cs));
            src = stg;
          }
          int rc = split_tokens(n_seq ? n_seq[m] : p->mu, p->T, src, p->tok_in + (size_t)tr * M, p->tok_tgt + (size_t)tr * M, cs);
          if (rc != PACI_OK) return rc;
          in = p->tok_in + (size_t)tr * M;
        } else {
          PACI_CUDA_OK(cudaStreamWaitEvent(cs, p->f_ready[(s - 1) * RING + r], 0));
          in = p->fbuf[(s - 1) * RING + r];
        }
        if (s == S - 1) {
          tgt = p->tok_tgt + (size_t)tr * M;
          outp = p->loss + m;
        } else {
          if (m >= RING) PACI_CUDA_OK(cudaStreamWaitEvent(cs, p->f_free[s * RING + r], 0));
          outp = p->fbuf[s * RING + r];
        }
        int rc = paci_forward_var(p->st[s], m, n_seq ? n_seq[m] : p->mu, in, tgt, outp, cs);
        if (rc != PACI_OK) return rc;   // EAGAIN cannot happen after the probe above
        if (s > 0) PACI_CUDA_OK(cudaEventRecord(p->f_free[(s - 1) * RING + r], cs));
        if (s < S - 1) PACI_CUDA_OK(cudaEventRecord(p->f_ready[s * RING + r], cs));
        nf[s] += 1;
        max_q[s] = std::max(max_q[s], (int)paci_unresolved(p->st[s]));
        if (s < S - 1) new_f[s + 1] += 1; else new_b[s] += 1;   // last stage: own loss is its backward input
        progressed = true;
      }
    }
    for (int s = 0; s < S; ++s) {
      vis_f[s] += new_f[s]; new_f[s] = 0;
      vis_b[s] += new_b[s]; new_b[s] = 0;
    }
    slots += 1;
    if (!progressed) return fail(PACI_ESTATE, "pipeline_run: schedule deadlock at slot %lld", (long long)slots);
  }
  for (int s = 0; s < S; ++s) {
    PACI_CUDA_OK(cudaEventRecord(p->ev_done[s], p->streams[s]));
    PACI_CUDA_OK(cudaStreamWaitEvent(p->main, p->ev_done[s], 0));
  }
  PACI_CUDA_OK(cudaEventRecord(p->ev_stop, p->main));
  if (rep->loss && n > 0)
    PACI_CUDA_OK(cudaMemcpyAsync(rep->loss, p->loss, (size_t)n * 4, cudaMemcpyDeviceToHost, p->main));
  PACI_CUDA_OK(cudaStreamSynchronize(p->main));
  PACI_CUDA_OK(cudaEventElapsedTime(&rep->elapsed_ms, p->ev_start, p->ev_stop));
  for (int s : {0, S - 1}) {                               // device-side validation of token / target ids
    int rc = paci_stage_check(p->st[s], p->main);
    if (rc != PACI_OK) return rc;
  }
  rep->n_slots = slots;
  rep->n_launches = paci_launch_count() - launches0;
  for (int s = 0; s < S; ++s) {
    if (rep->version) rep->version[s] = paci_version(p->st[s]);
    if (rep->max_q) rep->max_q[s] = max_q[s];
  }
  return PACI_OK;
}

}  // extern "C"
