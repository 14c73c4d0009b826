// Launch counter and per-kernel-class CUDA-event timing (cb_launch_count, cb_profile_begin/end).
// Instrumentation only: when profiling is off a ProfScope costs one atomic add.
#include "common.cuh"

#include <atomic>
#include <cstring>
#include <mutex>

namespace cb {

static const char* kNames[K_COUNT] = {"pack_weights", "conv_fwd", "pool_fwd", "conv_dgrad", "conv_wgrad", "wgrad_reduce", "pool_bwd", "head_misc",
                                      "logprob", "scan", "loss", "stats", "permutation", "sqnorm", "adam", "sample", "env_step"};
static std::atomic<uint64_t> g_launches{0};
static std::mutex g_mu;
static bool g_on = false; static int g_only = -1;
struct Rec { int cls; cudaEvent_t e0, e1; int n; double flops, bytes; };
static std::vector<Rec> g_recs;
static std::vector<cudaEvent_t> g_pool;

static cudaEvent_t get_event() {
  if (!g_pool.empty()) { cudaEvent_t e = g_pool.back(); g_pool.pop_back(); return e; }
  cudaEvent_t e; cudaEventCreate(&e); return e;
}

bool prof_active() { return g_on; }
void prof_add_launches(uint64_t n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

ProfScope::ProfScope(int cls, cudaStream_t s, int n, double flops, double bytes) : slot(-1), st(s) {
  g_launches.fetch_add((uint64_t)n, std::memory_order_relaxed);
  if (!g_on || (g_only >= 0 && g_only != cls)) return;
  std::lock_guard<std::mutex> lk(g_mu);
  Rec r{cls, get_event(), get_event(), n, flops, bytes};
  cudaEventRecord(r.e0, st);
  g_recs.push_back(r); slot = (int)g_recs.size() - 1;
}
ProfScope::~ProfScope() {
  if (slot < 0) return;
  std::lock_guard<std::mutex> lk(g_mu);
  cudaEventRecord(g_recs[slot].e1, st);
}

}  // namespace cb

using namespace cb;

extern "C" {

uint64_t cb_launch_count(void) { return g_launches.load(); }

int cb_profile_begin(int only_class) {
  std::lock_guard<std::mutex> lk(g_mu);
  for (Rec& r : g_recs) { g_pool.push_back(r.e0); g_pool.push_back(r.e1); }
  g_recs.clear(); g_on = true; g_only = only_class;
  return CB_OK;
}

int cb_profile_end(cb_prof_entry* out, int max) {
  CB_CUDA(cudaDeviceSynchronize());
  std::lock_guard<std::mutex> lk(g_mu);
  g_on = false;
  cb_prof_entry acc[K_COUNT]; memset(acc, 0, sizeof acc);
  for (Rec& r : g_recs) {
    float ms = 0.f; cudaEventElapsedTime(&ms, r.e0, r.e1);
    cb_prof_entry& a = acc[r.cls]; a.launches += (uint64_t)r.n; a.ms += ms; a.flops += r.flops; a.bytes += r.bytes;
    g_pool.push_back(r.e0); g_pool.push_back(r.e1);
  }
  g_recs.clear();
  int n = 0;
  for (int c = 0; c < K_COUNT && out && n < max; ++c)
    if (acc[c].launches) { out[n] = acc[c]; out[n].cls = c; strncpy(out[n].name, kNames[c], sizeof out[n].name - 1); ++n; }
  return n;
}

}  // extern "C"
