// Cleanba's actor/learner synchronisation on one GPU (Figure 1 right column PAPER.md:35-88, Table 1 PAPER.md:127-138,
// section 4.2, Synchronous variant PAPER.md:174).
//
// The paper runs an actor thread and a learner thread that hand each other work through two queues of maximum size 1; here the "threads"
// are two CUDA streams fed by ONE host thread, and each queue is a pair of device buffers whose hand-over is a CUDA event:
//   param_Q.put(pi_v)   = copy of the learner's parameters into actor slot v % 2 on the learner stream, then event param_ready[v % 2]
//   param_Q.get()       = the actor stream waits for that event (skipped at iteration 2: `if i != 2`, Figure 1 l.6-7)
//   data_Q.put(D_i)     = event data_ready[i % 2] on the actor stream after rollout i has filled data slot i % 2
//   data_Q.get()        = the learner stream waits for it;  put() blocking on a full queue = the actor stream waits for data_free[i % 2]
// so that the GPU runs rollout i+1 (policy pi_i) underneath learner iteration i (pi_i -> pi_{i+1} on D_i) exactly as Table 1 prescribes, and
// the Synchronous architecture (get() at every iteration) falls out as a flag.  Blocking never reaches the host: cb_pipeline_run only
// enqueues.  Actor and learner own separate cb_net objects (separate operand-layout weights and activations).
// Which policy produced which data is recorded ON THE DEVICE (version words travel with the parameter and data slots) and read back
// by cb_pipeline_records: the test compares them with Table 1.
#include "common.cuh"

namespace cb {

__global__ void tag_data_kernel(const int* __restrict__ param_version, int iteration, int* __restrict__ tag) { tag[0] = *param_version; tag[1] = iteration; }
__global__ void learner_log_kernel(const int* __restrict__ tag, int iteration, int* __restrict__ lver, int* __restrict__ rec, int* __restrict__ next_slot_version) {
  const int before = *lver;
  rec[0] = iteration; rec[1] = tag[0]; rec[2] = before; rec[3] = before + 1;
  *lver = before + 1; *next_slot_version = before + 1;
}
__global__ void set_int_kernel(int* p, int v) { *p = v; }

}  // namespace cb

using namespace cb;

struct cb_pipeline {
  cb_arch arch; cb_hparams hp; cb_pipeline_cfg cfg;
  cb_net *actor = nullptr, *learner = nullptr;
  size_t P = 0, frame = 0; int T = 0, B = 0, A = 0, n_upd = 1;
  float *params = nullptr, *adam_m = nullptr, *adam_v = nullptr; uint64_t opt_step = 0;
  float* aparams[2] = {nullptr, nullptr}; int* aver = nullptr;      // actor parameter slots and their device version words [2]
  int* lver = nullptr;                                              // learner's policy version (device)
  struct Slot { uint8_t* obs; int32_t* actions; float* rewards; uint8_t* dones; float* blogits; float* values; int* tag; } slot[2];
  uint8_t* cur[2] = {nullptr, nullptr}; int32_t* env_state = nullptr; int par = 0;
  float* stats = nullptr; int* log = nullptr; int cap = 64;
  cudaStream_t sa = nullptr, sl = nullptr;
  cudaEvent_t data_ready[2], data_free[2], param_ready[2], ev_start, ev_end, ev_join;
  int iter = 0; uint32_t gstep = 0;
  std::vector<void*> allocs;
};

#define PL_ALLOC(ptr, bytes) do { void* q__ = nullptr; cudaError_t e__ = cudaMalloc(&q__, (bytes) ? (bytes) : 16); if (e__ != cudaSuccess) { set_error("cudaMalloc of %zu bytes failed: %s", (size_t)(bytes), cudaGetErrorString(e__)); cb_pipeline_destroy(p); return CB_ENOMEM; } p->allocs.push_back(q__); (ptr) = (decltype(ptr))q__; } while (0)

extern "C" {

int cb_pipeline_policy_version(int sync, int iteration) {
  if (iteration < 1) return 0;
  return sync ? iteration : (iteration <= 2 ? 1 : iteration - 1);      // Table 1: Cleanba's actor uses pi_1, pi_1, pi_2, pi_3, ...
}

void cb_pipeline_destroy(cb_pipeline* p) {
  if (!p) return;
  cudaDeviceSynchronize();
  if (p->actor) cb_net_destroy(p->actor);
  if (p->learner) cb_net_destroy(p->learner);
  for (void* q : p->allocs) cudaFree(q);
  if (p->sa) {
    cudaStreamDestroy(p->sa); cudaStreamDestroy(p->sl);
    for (int i = 0; i < 2; ++i) { cudaEventDestroy(p->data_ready[i]); cudaEventDestroy(p->data_free[i]); cudaEventDestroy(p->param_ready[i]); }
    cudaEventDestroy(p->ev_start); cudaEventDestroy(p->ev_end); cudaEventDestroy(p->ev_join);
  }
  delete p;
}

int cb_pipeline_create(const cb_arch* arch, const cb_hparams* hp, const cb_pipeline_cfg* cfg, const float* params_dev, cb_pipeline** out) {
  if (out) *out = nullptr;
  if (!arch || !hp || !cfg || !params_dev || !out) { set_error("null argument"); return CB_EINVAL; }
  if (hp->T < 1 || hp->B < 1) { set_error("T and B must be positive"); return CB_EINVAL; }
  cb_pipeline* p = new (std::nothrow) cb_pipeline();
  if (!p) { set_error("out of host memory"); return CB_ENOMEM; }
  p->arch = *arch; p->hp = *hp; p->cfg = *cfg; p->T = hp->T; p->B = hp->B; p->A = arch->n_actions;
  p->frame = (size_t)arch->in_c * arch->in_h * arch->in_w;
  p->n_upd = hp->algo == CB_ALGO_PPO ? hp->epochs * hp->minibatches : (hp->minibatches < 1 ? 1 : hp->minibatches);
  int rc;
  if ((rc = cb_net_create(arch, hp->B, &p->actor)) || (rc = cb_net_create(arch, (hp->T + 1) * hp->B, &p->learner))) { cb_pipeline_destroy(p); return rc; }
  p->P = cb_param_count(p->learner);
  const int T = p->T, B = p->B, A = p->A; const size_t P4 = p->P * 4;
  PL_ALLOC(p->params, P4); PL_ALLOC(p->adam_m, P4); PL_ALLOC(p->adam_v, P4); PL_ALLOC(p->aparams[0], P4); PL_ALLOC(p->aparams[1], P4);
  PL_ALLOC(p->aver, 16); PL_ALLOC(p->lver, 16);
  for (int s = 0; s < 2; ++s) {
    cb_pipeline::Slot& d = p->slot[s];
    PL_ALLOC(d.obs, (size_t)(T + 1) * B * p->frame); PL_ALLOC(d.actions, (size_t)T * B * 4); PL_ALLOC(d.rewards, (size_t)T * B * 4); PL_ALLOC(d.dones, (size_t)T * B);
    PL_ALLOC(d.blogits, (size_t)T * B * A * 4); PL_ALLOC(d.values, (size_t)(T + 1) * B * 4); PL_ALLOC(d.tag, 16);
    PL_ALLOC(p->cur[s], (size_t)B * p->frame);
  }
  PL_ALLOC(p->env_state, (size_t)B * cb_env_state_ints() * 4);
  PL_ALLOC(p->stats, (size_t)p->cap * p->n_upd * CB_N_STATS * 4); PL_ALLOC(p->log, (size_t)p->cap * 4 * 4);
  CB_CUDA(cudaStreamCreateWithFlags(&p->sa, cudaStreamNonBlocking)); CB_CUDA(cudaStreamCreateWithFlags(&p->sl, cudaStreamNonBlocking));
  for (int i = 0; i < 2; ++i) {
    CB_CUDA(cudaEventCreateWithFlags(&p->data_ready[i], cudaEventDisableTiming)); CB_CUDA(cudaEventCreateWithFlags(&p->data_free[i], cudaEventDisableTiming));
    CB_CUDA(cudaEventCreateWithFlags(&p->param_ready[i], cudaEventDisableTiming));
  }
  CB_CUDA(cudaEventCreate(&p->ev_start)); CB_CUDA(cudaEventCreate(&p->ev_end)); CB_CUDA(cudaEventCreateWithFlags(&p->ev_join, cudaEventDisableTiming));
  // pi_1: the learner's parameters, zero optimizer state; main thread's `param_Q.put(agent.param)` (Figure 1 l.15-16) fills actor slot 1
  CB_CUDA(cudaMemcpyAsync(p->params, params_dev, P4, cudaMemcpyDeviceToDevice, p->sl));
  CB_CUDA(cudaMemsetAsync(p->adam_m, 0, P4, p->sl)); CB_CUDA(cudaMemsetAsync(p->adam_v, 0, P4, p->sl));
  CB_CUDA(cudaMemsetAsync(p->stats, 0, (size_t)p->cap * p->n_upd * CB_N_STATS * 4, p->sl)); CB_CUDA(cudaMemsetAsync(p->log, 0, (size_t)p->cap * 16, p->sl));
  CB_CUDA(cudaMemcpyAsync(p->aparams[1], p->params, P4, cudaMemcpyDeviceToDevice, p->sl));
  set_int_kernel<<<1, 1, 0, p->sl>>>(p->lver, 1); set_int_kernel<<<1, 1, 0, p->sl>>>(p->aver + 1, 1); set_int_kernel<<<1, 1, 0, p->sl>>>(p->aver, 0);
  CB_CUDA(cudaGetLastError());
  CB_CUDA(cudaEventRecord(p->param_ready[1], p->sl));
  // s_next = E.reset() (Alg. 1 l.3)
  if ((rc = launch_env_reset(cfg->env_seed, B, arch->in_c, arch->in_h, arch->in_w, p->env_state, p->cur[0], p->sa))) { cb_pipeline_destroy(p); return rc; }
  CB_CUDA(cudaDeviceSynchronize());
  *out = p;
  return CB_OK;
}

int cb_pipeline_run(cb_pipeline* p, int iterations) {
  if (!p || iterations < 0) { set_error("bad argument"); return CB_EINVAL; }
  if (iterations == 0) return CB_OK;
  const int T = p->T, B = p->B, A = p->A, prec = p->hp.precision; int rc;
  const bool sync = p->cfg.sync != 0, serial = p->cfg.serial != 0;
  // the timed region starts when BOTH streams have drained their earlier work
  CB_CUDA(cudaEventRecord(p->ev_join, p->sl)); CB_CUDA(cudaStreamWaitEvent(p->sa, p->ev_join, 0)); CB_CUDA(cudaEventRecord(p->ev_start, p->sa));
  CB_CUDA(cudaStreamWaitEvent(p->sl, p->ev_start, 0));
  for (int n = 0; n < iterations; ++n) {
    const int i = ++p->iter, ds = i & 1;
    cb_pipeline::Slot& d = p->slot[ds];
    // ---------------- actor (Figure 1 right, l.4-10) ----------------
    const int v = cb_pipeline_policy_version(sync, i), ps = v & 1;
    if (sync || i != 2) CB_CUDA(cudaStreamWaitEvent(p->sa, p->param_ready[ps], 0));        // params = param_Q.get()
    if (i > 2) CB_CUDA(cudaStreamWaitEvent(p->sa, p->data_free[ds], 0));                   // data_Q.put blocks while the slot is still being learnt from
    tag_data_kernel<<<1, 1, 0, p->sa>>>(p->aver + ps, i, d.tag);
    CB_CUDA(cudaMemcpyAsync(d.obs, p->cur[p->par], (size_t)B * p->frame, cudaMemcpyDeviceToDevice, p->sa));      // o_0 = s_next of the previous rollout (Alg. 1 l.7)
    for (int t = 0; t < T; ++t) {                                                           // rollout(params, batch_size): Alg. 1 l.6-10
      if ((rc = cb_policy_forward(p->actor, t == 0 ? p->aparams[ps] : nullptr, p->cur[p->par], B, p->cfg.sample_seed, (uint64_t)p->gstep, 0u, prec,
                                  d.blogits + (size_t)t * B * A, d.values + (size_t)t * B, d.actions + (size_t)t * B, p->sa)) < 0) return rc;
      if ((rc = launch_env_step(p->cfg.env_seed, B, p->arch.in_c, p->arch.in_h, p->arch.in_w, p->gstep, d.actions + (size_t)t * B, p->env_state, p->cur[p->par],
                                d.obs + (size_t)(t + 1) * B * p->frame, p->cur[p->par ^ 1], d.rewards + (size_t)t * B, d.dones + (size_t)t * B, p->sa))) return rc;
      p->par ^= 1; p->gstep += 1;
    }
    if (p->cfg.actor_values)                                                                // v_next of Alg. 1 l.11, with the rollout's parameters
      if ((rc = cb_policy_forward(p->actor, nullptr, p->cur[p->par], B, 0, 0, 0u, prec, nullptr, d.values + (size_t)T * B, nullptr, p->sa)) < 0) return rc;
    CB_CUDA(cudaEventRecord(p->data_ready[ds], p->sa));                                     // data_Q.put(data)
    if (serial) CB_CUDA(cudaDeviceSynchronize());
    // ---------------- learner (Figure 1 right, l.11-14) ----------------
    CB_CUDA(cudaStreamWaitEvent(p->sl, p->data_ready[ds], 0));                              // data = data_Q.get()
    float* srow = p->stats + (size_t)((i - 1) % p->cap) * p->n_upd * CB_N_STATS;
    if ((rc = cb_learner_step(p->learner, p->params, p->adam_m, p->adam_v, &p->opt_step, d.obs, d.actions, d.rewards, d.dones, d.blogits,
                              p->cfg.actor_values ? d.values : nullptr, &p->hp, srow, p->sl)) < 0) return rc;      // agent.learn(data)
    const int ns = (i + 1) & 1;                                                             // param_Q.put(agent.param): pi_{i+1} -> actor slot (i+1) % 2
    learner_log_kernel<<<1, 1, 0, p->sl>>>(d.tag, i, p->lver, p->log + (size_t)((i - 1) % p->cap) * 4, p->aver + ns);
    CB_CUDA(cudaMemcpyAsync(p->aparams[ns], p->params, p->P * 4, cudaMemcpyDeviceToDevice, p->sl));
    CB_CUDA(cudaEventRecord(p->param_ready[ns], p->sl));
    CB_CUDA(cudaEventRecord(p->data_free[ds], p->sl));
    CB_CUDA(cudaGetLastError());
    if (serial) CB_CUDA(cudaDeviceSynchronize());
  }
  CB_CUDA(cudaEventRecord(p->ev_join, p->sa)); CB_CUDA(cudaStreamWaitEvent(p->sl, p->ev_join, 0)); CB_CUDA(cudaEventRecord(p->ev_end, p->sl));
  return CB_OK;
}

int cb_pipeline_wait(cb_pipeline* p, float* elapsed_ms) {
  if (!p) { set_error("null argument"); return CB_EINVAL; }
  int rc;
  if ((rc = cb_check_errors(p->actor, p->sa))) return rc;
  if ((rc = cb_check_errors(p->learner, p->sl))) return rc;
  if (elapsed_ms) { *elapsed_ms = 0.f; if (p->iter > 0) CB_CUDA(cudaEventElapsedTime(elapsed_ms, p->ev_start, p->ev_end)); }
  return CB_OK;
}

int cb_pipeline_state(cb_pipeline* p, float** params, float** adam_m, float** adam_v, uint64_t* opt_step, int* iterations) {
  if (!p) { set_error("null argument"); return CB_EINVAL; }
  if (params) *params = p->params; if (adam_m) *adam_m = p->adam_m; if (adam_v) *adam_v = p->adam_v;
  if (opt_step) *opt_step = p->opt_step; if (iterations) *iterations = p->iter;
  return CB_OK;
}

int cb_pipeline_records(cb_pipeline* p, cb_pipeline_record* out, int max) {
  if (!p || !out || max < 0) { set_error("bad argument"); return CB_EINVAL; }
  int rc = cb_pipeline_wait(p, nullptr); if (rc) return rc;
  const int n = std::min(std::min(p->iter, p->cap), max), first = p->iter - n;      // the last n iterations
  std::vector<int> host((size_t)p->cap * 4);
  CB_CUDA(cudaMemcpy(host.data(), p->log, host.size() * 4, cudaMemcpyDeviceToHost));
  for (int k = 0; k < n; ++k) {
    const int* r = &host[(size_t)((first + k) % p->cap) * 4];
    out[k].iteration = r[0]; out[k].data_policy_version = r[1]; out[k].learner_version_before = r[2]; out[k].learner_version_after = r[3];
  }
  return n;
}

int cb_pipeline_rollout(cb_pipeline* p, int iteration, const uint8_t** obs, const int32_t** actions, const float** rewards, const uint8_t** dones,
                        const float** behaviour_logits, const float** values, const float** stats) {
  if (!p || iteration < 1 || iteration > p->iter || iteration <= p->iter - 2) { set_error("only the data slots of the last two iterations exist"); return CB_EINVAL; }
  const cb_pipeline::Slot& d = p->slot[iteration & 1];
  if (obs) *obs = d.obs; if (actions) *actions = d.actions; if (rewards) *rewards = d.rewards; if (dones) *dones = d.dones;
  if (behaviour_logits) *behaviour_logits = d.blogits; if (values) *values = d.values;
  if (stats) *stats = p->stats + (size_t)((iteration - 1) % p->cap) * p->n_upd * CB_N_STATS;
  return CB_OK;
}

}  // extern "C"
