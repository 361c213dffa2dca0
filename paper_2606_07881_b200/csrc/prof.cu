// prof.cu -- in-library sampled kernel timing (bench.py's "roofline" object).
// Every top-level launcher opens a ProfScope with its category and its ALGORITHMIC work (flops,
// bytes).  All launches are counted; every `stride`-th one is bracketed by a pair of CUDA events
// recorded on the stream the kernel is launched on, so the measurement lives inside the timed
// region of the benchmark at negligible cost.  Host code only.
//
// Exclusive samples.  The schedule driver runs the S emulated stages on S streams, so a kernel bracketed
// by events on its own stream shares the SMs with the other stages' kernels and its event time is a
// latency under contention, not its own duration.  While a pipeline run is active (prof_set_peer_streams)
// a SAMPLED launch therefore first waits for everything already queued on the other stage streams, and
// those streams wait for the sample's end event: the sampled kernel runs alone, with the caches and clocks
// of the real step, and 1 launch in `stride` pays for it.
#include <mutex>
#include <vector>

#include "common.cuh"

namespace paci {

namespace {
struct Sample { int cat; double flops, bytes; cudaEvent_t e0, e1; };
std::mutex g_mu;
int g_stride = 0;
int64_t g_counter = 0;
paci_prof_entry g_tot[PACI_PROF_NCAT];
std::vector<Sample> g_samples;
std::vector<cudaEvent_t> g_pool;
size_t g_pool_used = 0;
std::vector<cudaStream_t> g_peers;

cudaEvent_t take_event() {
  if (g_pool_used == g_pool.size()) {
    cudaEvent_t e;
    if (cudaEventCreate(&e) != cudaSuccess) return nullptr;
    g_pool.push_back(e);
  }
  return g_pool[g_pool_used++];
}
const char* const kNames[PACI_PROF_NCAT] = {
    "gemm_fwd", "gemm_dgrad", "gemm_wgrad", "attention_fwd", "attention_bwd", "layernorm_fwd", "layernorm_bwd",
    "gelu_fwd", "gelu_bwd", "colsum", "embedding", "softmax_ce", "adamw", "other", "gemm_bwd_pair"};
}  // namespace

ProfScope::ProfScope(int cat, double flops, double bytes, cudaStream_t s) : idx_(-1), stream_(s) {
  if (g_stride <= 0) return;
  std::lock_guard<std::mutex> g(g_mu);
  paci_prof_entry& t = g_tot[cat];
  t.launches += 1; t.flops += flops; t.bytes += bytes;
  if (g_counter++ % g_stride != 0) return;
  Sample smp{cat, flops, bytes, take_event(), take_event()};
  if (!smp.e0 || !smp.e1) return;
  for (cudaStream_t peer : g_peers) {
    if (peer == s) continue;
    cudaEvent_t e = take_event();
    if (!e || cudaEventRecord(e, peer) != cudaSuccess || cudaStreamWaitEvent(s, e, 0) != cudaSuccess) return;
  }
  if (cudaEventRecord(smp.e0, s) != cudaSuccess) return;
  g_samples.push_back(smp);
  idx_ = (int)g_samples.size() - 1;
}
ProfScope::~ProfScope() {
  if (idx_ < 0) return;
  std::lock_guard<std::mutex> g(g_mu);
  cudaEventRecord(g_samples[idx_].e1, stream_);
  for (cudaStream_t peer : g_peers)
    if (peer != stream_) cudaStreamWaitEvent(peer, g_samples[idx_].e1, 0);
}

void prof_set_peer_streams(const cudaStream_t* streams, int n) {
  std::lock_guard<std::mutex> g(g_mu);
  g_peers.assign(streams, streams + (streams ? n : 0));
}

}  // namespace paci

using namespace paci;

extern "C" {

int paci_profile_begin(int32_t sample_stride) {
  std::lock_guard<std::mutex> g(g_mu);
  g_stride = sample_stride > 0 ? sample_stride : 0;
  g_counter = 0;
  g_samples.clear();
  g_pool_used = 0;
  for (auto& t : g_tot) t = paci_prof_entry{};
  return PACI_OK;
}

int paci_profile_end(paci_prof_entry* out) {
  PACI_CUDA_OK(cudaDeviceSynchronize());
  std::lock_guard<std::mutex> g(g_mu);
  g_stride = 0;
  for (const Sample& s : g_samples) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, s.e0, s.e1) != cudaSuccess) continue;
    paci_prof_entry& t = g_tot[s.cat];
    t.sampled += 1; t.sampled_flops += s.flops; t.sampled_bytes += s.bytes; t.sampled_ms += ms;
  }
  if (out) for (int i = 0; i < PACI_PROF_NCAT; ++i) out[i] = g_tot[i];
  g_samples.clear();
  g_pool_used = 0;
  return PACI_OK;
}

const char* paci_profile_category_name(int32_t cat) {
  return (cat >= 0 && cat < PACI_PROF_NCAT) ? kNames[cat] : "";
}

}  // extern "C"
