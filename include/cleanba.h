/* =============================================================================================
 * cleanba.h -- C ABI of the B200-native hot path of Cleanba's actor-learner method
 * (arXiv 2310.00036).  Citations are PAPER.md:<line> or a reading "A<n>" of DESIGN.md section 3.
 *
 * The path (Algorithm 1): batched policy/value inference on stacked
 * 84x84x4 uint8 frames with categorical sampling (l.8), and the learner step (l.11-20): network
 * forward, V-trace or GAE targets, IMPALA or clipped-PPO loss (Eq. 2-3),
 * backward, global grad-norm clip and Adam.
 *
 * Conventions for EVERY entry point:
 *   - "dev" pointers are CUDA device pointers, "host" pointers are host pointers.  The caller
 *     owns every buffer it passes; the library owns only the workspace inside cb_net.
 *   - All arrays are dense row-major, last index fastest; trajectories are time-major [T,B,...]
 *     exactly as the paper stores D.
 *   - All work is enqueued on `stream` (a cudaStream_t passed as void*; NULL = legacy default
 *     stream).  No call synchronises the device except where stated (workspace growth).
 *   - Return value: 0 (CB_OK) or a negative code; cb_last_error() gives the text of the last
 *     failure on the calling thread.  Nothing aborts or throws.
 *   - Determinism (A16): identical inputs give bitwise identical outputs (fixed-order
 *     reductions, no floating-point atomics).
 * ============================================================================================= */
#ifndef CLEANBA_H_
#define CLEANBA_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { CB_OK = 0, CB_EINVAL = -1, CB_ENOMEM = -2, CB_ECUDA = -3 };
enum { CB_ARCH_NATURE = 0, CB_ARCH_IMPALA = 1 };
enum { CB_PREC_FP32_REF = 0, CB_PREC_BF16_TC = 1 };
enum { CB_ALGO_IMPALA = 0, CB_ALGO_PPO = 1 };
/* stats record per gradient update: loss, pg_loss, v_loss, entropy, grad_norm (pre-clip),
 * approx_kl, clip_frac (PPO), mean_rho (IMPALA); unused fields are 0. */
enum { CB_N_STATS = 8 };

/* Network description.  kind 0 = Nature-CNN (BASELINE.json configs[0]): conv 8x8s4, 4x4s2,
 * 3x3s1 (VALID), fc, heads.  kind 1 = IMPALA-ResNet: 3 x [conv3x3 pad 1,
 * max-pool 3x3 s2 SAME (A10), 2 residual blocks], ReLU, fc, ReLU, policy + value heads.
 * Input is in_c x in_h x in_w uint8 (4 x 84 x 84). */
typedef struct {
  int kind;
  int in_c, in_h, in_w;
  int channels[3];
  int fc;
  int n_actions; /* 18 */
} cb_arch;

/* Hyper-parameters of one learner call (Tables 2-3; A12 for Adam). */
typedef struct {
  int algo;      /* CB_ALGO_* */
  int precision; /* CB_PREC_* */
  int T, B;      /* unroll length, envs */
  float gamma, lambda_;             /* V-trace lambda (1) or GAE lambda (0.95) */
  float rho_bar, c_bar, rho_pg_bar; /* IMPALA */
  float clip_eps;                   /* PPO */
  int epochs, minibatches, norm_adv; /* PPO.  IMPALA: minibatches = number of env groups (A21,
                                      * PAPER.md:213, 401): each group of B/minibatches whole trajectories is one update */
  uint64_t perm_seed;               /* PPO minibatch permutation (A17) */
  float vf_coef, ent_coef;          /* c1, c2 */
  float lr, beta1, beta2, adam_eps, max_grad_norm;
  int loss_reduction;               /* 0 = mean over samples, 1 = sum (A4) */
  int optimizer;                    /* 0 = Adam (A12), 1 = RMSprop (Table 3; A22): state in adam_v only */
  float rms_decay, rms_eps;         /* 0.99, 0.01; eps sits inside the square root */
} cb_hparams;

typedef struct cb_net cb_net; /* opaque: layer table, parameter offsets, device workspaces */

/* ---- lifetime -------------------------------------------------------------------------- */
/* Builds the layer table for `arch`.  max_frames is a hint: the device workspace for
 * `max_frames` frames is allocated lazily (cudaMalloc) on the first forward/learner call in a
 * given precision and grown if a later call needs more (growth synchronises the device).
 * Needs no GPU.  *out is NULL on failure. */
int cb_net_create(const cb_arch* arch, int max_frames, cb_net** out);
void cb_net_destroy(cb_net* net);

/* P = number of fp32 parameters.  Canonical flat order: layer order, weight
 * then bias; conv weights [Cout,Cin,kh,kw]; fc weights [out,in] with `in` flattened (C,H,W);
 * then pi.w [A,fc], pi.b [A], v.w [fc], v.b [1]. */
size_t cb_param_count(const cb_net* net);
/* Tensor i of that order: name (static string), offset in elements, rank and dims (<= 4).
 * Returns CB_EINVAL past the last tensor. */
int cb_param_layout(const cb_net* net, int i, const char** name, size_t* offset, int* rank, int dims[4]);

/* He-normal initialisation on the HOST (A14): weights N(0, 2/fan_in), biases 0, Philox4x32-10 +
 * Box-Muller in fp64; deterministic in `seed`.  params_host: host [P], written. */
int cb_net_init(const cb_net* net, uint64_t seed, float* params_host);

/* ---- actor side (Alg. 1 l.8) ------------------------------------------------ */
/* logits, value = net(obs);  actions[b] = argmax_i(logits[b,i] + Gumbel_i), the Gumbel noise
 * from Philox4x32-10 with key = seed and counter = (env_offset + b, step_lo, step_hi, i/4), word
 * i%4 (A9).  params: dev [P] fp32 (16-byte aligned), or NULL to reuse the operand-layout weights packed by the previous
 * call on this net in the same precision mode (an actor takes new parameters from its queue once
 * per rollout, not per step: Figure 1 / PAPER.md:148-150; CB_EINVAL if there was no such call, or if a learner
 * call has run on this net since).  obs: dev uint8 [B,in_c,in_h,in_w], 4-byte aligned.  precision: CB_PREC_*.
 * Outputs (dev): logits fp32 [B,A], value fp32 [B], actions int32 [B]; any may be NULL.
 * Launch behaviour: from the third call with the same (precision, B, obs pointer) on, the network
 * trunk is replayed as a CUDA graph on `stream` (captured on a library-owned stream during the
 * second call); the frames are read from `obs` at replay time, so a rollout loop should reuse its
 * observation buffers.  Results are bitwise those of the direct launches. */
int cb_policy_forward(cb_net* net, const float* params, const uint8_t* obs, int B, uint64_t seed,
                      uint64_t step, uint32_t env_offset, int precision, float* logits, float* value,
                      int32_t* actions, void* stream);

/* ---- learner side (Alg. 1 l.11-20) -------------------------------------- */
/* One learner call: IMPALA = `minibatches` V-trace gradient updates, one per group of envs in order (1 = one
 * full-batch update); PPO = GAE, then epochs x minibatches updates over a seeded permutation (epoch e of this call
 * uses permutation epoch (*opt_step at entry / minibatches) + e, A23).  Updated in place (dev fp32 [P]): params,
 * adam_m, adam_v.
 * opt_step: host counter, incremented once per gradient update (Adam's k, from 1).
 * obs: dev uint8 [T+1,B,in_c,in_h,in_w], 4-byte aligned; actions: dev int32 [T,B], each in [0, A) (an out-of-range action is
 * clamped into range by the kernels that index with it, never read out of bounds); rewards: dev fp32 [T,B];
 * dones: dev uint8 [T,B], 1 <=> the step taken at t ended the episode (A1);
 * behaviour_logits: dev fp32 [T,B,A];
 * behaviour_values: dev fp32 [T+1,B] or NULL.  PPO only (A3b; Alg. 1 l.8-12): the values the actor
 * computed at rollout time (v_t for t < T, v_next for the bootstrap observation); GAE uses them and the learner's
 * iteration-start forward over (T+1)B frames is skipped.  NULL = recompute them with the iteration-start parameters
 * (A3).  IMPALA ignores it (V-trace is defined on the current parameters' values).
 * stats: dev fp32 [n_updates, CB_N_STATS], written.
 * Returns the number of gradient updates done (> 0) or a negative error.
 * A cb_net is a single-stream, single-role object: calls on one net must not overlap in time, and after a learner
 * call the operand-layout weights of that precision mode are stale, so cb_policy_forward(params = NULL) fails until
 * parameters are passed again.  An actor running concurrently with the learner uses its own cb_net (cb_pipeline). */
int cb_learner_step(cb_net* net, float* params, float* adam_m, float* adam_v, uint64_t* opt_step,
                    const uint8_t* obs, const int32_t* actions, const float* rewards,
                    const uint8_t* dones, const float* behaviour_logits, const float* behaviour_values,
                    const cb_hparams* hp, float* stats, void* stream);

/* The same call in three parts, for a data-parallel learner (every device
 * runs Alg. 1 on its own envs and "the gradient of the copies" is averaged before the optimizer step):
 *   n = cb_learner_begin(...)                validates, keeps the pointers, does the per-call work (PPO: values, GAE,
 *                                            permutations); returns the number of updates n
 *   for u in 0..n-1:
 *     cb_learner_grad(net, u, &g, stream)    forward, targets/loss, backward of update u with the CURRENT params;
 *                                            *g = library-owned dev fp32 [P] gradient (pre-clip), written stats row u
 *     ... the caller may replace *g by the average over ranks here (in place, on `stream`) ...
 *     cb_learner_apply(net, u, stream)       global-norm clip + optimizer on *g; increments *opt_step
 * All pointers passed to cb_learner_begin must stay valid until the last cb_learner_apply.  Updates must be taken in
 * order, each grad followed by its apply.  cb_learner_step is exactly this sequence. */
int cb_learner_begin(cb_net* net, float* params, float* adam_m, float* adam_v, uint64_t* opt_step,
                     const uint8_t* obs, const int32_t* actions, const float* rewards,
                     const uint8_t* dones, const float* behaviour_logits, const float* behaviour_values,
                     const cb_hparams* hp, float* stats, void* stream);
int cb_learner_grad(cb_net* net, int update, float** grad_dev, void* stream);
int cb_learner_apply(cb_net* net, int update, void* stream);

/* Fixed-order sum over ranks for the gradient exchange of a data-parallel learner: out[i] = scale * (in[0][i] + in[1][i]
 * + ... + in[G-1][i]) added in rank order (bitwise the same on every rank that holds the same G slices).  in: dev fp32
 * [G, n] (slice r = what rank r contributed); out: dev fp32 [n], may alias in[0].  16-byte loads when n % 4 == 0 and the
 * buffers are 16-byte aligned, scalar otherwise (same bits). */
int cb_sum_ranks(const float* in, int G, size_t n, float scale, float* out, void* stream);

/* Asynchronous errors.  A tcgen05 pipeline wait that times out inside a kernel (bounded spin: a lost arrival must not
 * hang the GPU) sets a device flag; the step's optimizer then leaves params / optimizer state untouched and the
 * stats row reads NaN (cb_learner_*), logits / value read NaN and actions -1 (cb_policy_forward), and a host-visible
 * word is set.  Every later call on the net, and cb_check_errors, return CB_ECUDA once and clear the condition.
 * cb_check_errors synchronises `stream` first, so after it returns CB_OK the results of all earlier calls are valid. */
int cb_check_errors(cb_net* net, void* stream);
/* Test hook: raises that device flag in `precision` mode as a timed-out kernel would (enqueued on `stream`). */
int cb_debug_inject_timeout(cb_net* net, int precision, void* stream);

/* Device pointers to the library-owned results of the LAST cb_learner_step (valid until the next
 * call on this net): which = 0: forward logits fp32 [(T+1)B, A+1] (column A is the value), from the
 * first forward (CB_EINVAL when PPO was given behaviour_values: no such forward ran); 1: vs (IMPALA) or advantages (PPO) fp32 [T,B]; 2: pg advantages (IMPALA) or returns
 * (PPO) fp32 [T,B]; 3: gradient of the last update before clipping, fp32 [P]. */
int cb_learner_view(const cb_net* net, int which, const void** dev_ptr, size_t* count);

/* ---- the path's sub-steps, exposed one by one (all dev pointers, fp32 unless noted) -------- */
/* A9: Gumbel-max sampling from given logits [B,A] -> actions int32 [B]. */
int cb_sample_actions(const float* logits, int B, int A, uint64_t seed, uint64_t step,
                      uint32_t env_offset, int32_t* actions, void* stream);
/* O2: log-softmax of logits [N, ld] (first A columns) -> logp_a [N] = log pi(actions[n]), entropy [N]
 * (nullable). */
int cb_logprob_entropy(const float* logits, int ld, int N, int A, const int32_t* actions, float* logp_a,
                       float* entropy, void* stream);
/* O4 V-trace (A2): V [T+1,B]; r, logpi, logmu [T,B]; d uint8 [T,B] -> vs, pgadv, rho [T,B]
 * (rho nullable).  One lane per env, reverse-time scan. */
int cb_vtrace(int T, int B, const float* V, const float* r, const uint8_t* d, const float* logpi,
              const float* logmu, float gamma, float lambda_, float rho_bar, float c_bar,
              float rho_pg_bar, float* vs, float* pgadv, float* rho, void* stream);
/* O6 GAE (A3): -> adv, ret [T,B]. */
int cb_gae(int T, int B, const float* V, const float* r, const uint8_t* d, float gamma, float lambda_,
           float* adv, float* ret, void* stream);
/* O5 / O7: the loss of one update with its adjoint seeds (a8).  head: dev fp32 [N, A+1] (A logits, then the value); dhead: dev
 * [N, A+1] in the precision mode's storage type (fp32 / bf16) = dL/dlogits, dL/dV; stats: dev fp32 [CB_N_STATS] (slot 4, the
 * gradient norm, is left 0); scratch: dev, >= cb_loss_scratch_bytes(N) bytes.  IMPALA (A4-A6): vs, pgadv, rho [N] from cb_vtrace.
 * PPO (Eq. 2-3; A5-A8): sample n of the minibatch is row idx[n] (idx NULL: n) of actions / adv / ret / logp_old
 * while head row n is the minibatch's own forward; norm_adv = per-minibatch advantage normalisation. */
size_t cb_loss_scratch_bytes(int N);
int cb_impala_loss(int N, int A, const float* head, const int32_t* actions, const float* vs, const float* pgadv, const float* rho,
                   float vf_coef, float ent_coef, int loss_reduction, int precision, void* dhead, float* stats, void* scratch,
                   void* stream);
int cb_ppo_loss(int m, int A, const float* head, const int32_t* idx, const int32_t* actions, const float* adv, const float* ret,
                const float* logp_old, float clip_eps, float vf_coef, float ent_coef, int norm_adv, int precision, void* dhead,
                float* stats, void* scratch, void* stream);
/* A17: Fisher-Yates permutation of N indices for (seed, epoch) -> perm int32 [N]. */
int cb_permutation(uint64_t seed, uint32_t epoch, int N, int32_t* perm, void* stream);
/* The same with caller-provided scratch (dev uint32 [N]), so that no allocation happens inside the call. */
int cb_permutation_ws(uint64_t seed, uint32_t epoch, int N, int32_t* perm, uint32_t* scratch, void* stream);
/* The same for callers that may not allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc): the scratch
 * is a static device array of CB_PERM_STATIC_MAX draws (256 KiB held by every GPU that loads the library, until exit); the call
 * performs no cudaMalloc / cudaFree.  perm: dev int32 [N], written; N > CB_PERM_STATIC_MAX -> CB_EINVAL (use cb_permutation_ws).
 * All calls on a device share the array: calls that overlap on the GPU (other streams, concurrent graph replays) race; calls
 * ordered on one stream are safe, and no state carries from one call to the next (every draw is written before it is read). */
#define CB_PERM_STATIC_MAX 65536
int cb_permutation_static(uint64_t seed, uint32_t epoch, int N, int32_t* perm, void* stream);
/* O9 (A12, A13): global-norm clip + Adam over flat fp32 buffers of P elements (16-byte aligned);
 * k = update count (from 1).  grad_norm: dev fp32 [1], written (pre-clip norm; nullable).
 * scratch: dev, at least cb_clip_adam_scratch_bytes(P) bytes. */
size_t cb_clip_adam_scratch_bytes(size_t P);
int cb_clip_adam(size_t P, float* params, float* adam_m, float* adam_v, const float* grad, uint64_t k,
                 float lr, float beta1, float beta2, float eps, float max_norm, float* grad_norm,
                 void* scratch, void* stream);

/* ---- Cleanba's actor/learner architecture on one GPU ------------------------ */
/* Figure 1 right column, Table 1, section 4.2: an actor and a learner
 * exchange parameters and rollouts through two queues of size 1, the actor skipping param_Q.get() at iteration 2, so that from
 * iteration 3 on the learner trains pi_i on the rollout of pi_{i-1} while the actor already collects the rollout of pi_i.  Here
 * the two threads are two CUDA streams and each queue is a double buffer handed over by a CUDA event (csrc/pipeline.cu); the
 * environment is a seeded synthetic stepper on the device (cb_env_*; definition: synth.py BlobEnv).  sync = 1 gives the
 * Synchronous architecture ("commenting out line 7").  All buffers are library-owned. */
typedef struct {
  int sync;          /* 0 = Cleanba's architecture, 1 = Synchronous architecture (Table 1) */
  int actor_values;  /* PPO: hand the learner the values the actor computed at rollout time (A3b) */
  int serial;        /* 1 = synchronise the device after every rollout and every learner call (reference execution for tests) */
  uint64_t env_seed, sample_seed;
} cb_pipeline_cfg;
/* iteration i of the learner: the policy version whose rollout it trained on, and its own version before / after -- written by
 * the device in stream order (Table 1: Cleanba 1:(1,1->2), 2:(1,2->3), 3:(2,3->4), ...; Synchronous i:(i,i->i+1)). */
typedef struct { int iteration, data_policy_version, learner_version_before, learner_version_after; } cb_pipeline_record;
typedef struct cb_pipeline cb_pipeline;
/* hp: algo, precision, T, B and the loss / optimizer settings of every learner call.  params: dev fp32 [P], copied (pi_1). */
int cb_pipeline_create(const cb_arch* arch, const cb_hparams* hp, const cb_pipeline_cfg* cfg, const float* params, cb_pipeline** out);
void cb_pipeline_destroy(cb_pipeline* p);
/* Enqueues `iterations` more iterations (one rollout of T steps on B envs + one learner call each) and returns without waiting. */
int cb_pipeline_run(cb_pipeline* p, int iterations);
/* Waits for both streams; CB_ECUDA if a kernel reported an asynchronous error.  elapsed_ms (nullable): device time of the last
 * cb_pipeline_run, from both streams idle to both streams done. */
int cb_pipeline_wait(cb_pipeline* p, float* elapsed_ms);
/* Library-owned learner state (dev fp32 [P] each), the update count and the iterations enqueued so far; any may be NULL. */
int cb_pipeline_state(cb_pipeline* p, float** params, float** adam_m, float** adam_v, uint64_t* opt_step, int* iterations);
/* The records of the last min(iterations, 64, max) iterations, oldest first; waits first.  Returns how many were written. */
int cb_pipeline_records(cb_pipeline* p, cb_pipeline_record* out, int max);
/* Device pointers of the rollout storage D of `iteration` (one of the last two): obs uint8 [T+1,B,C,H,W], actions
 * int32 [T,B], rewards fp32 [T,B], dones uint8 [T,B], behaviour_logits fp32 [T,B,A], values fp32 [T+1,B] (row T only with
 * actor_values), and the stats rows [n_updates, CB_N_STATS] of that iteration's learner call.  Any may be NULL. */
int cb_pipeline_rollout(cb_pipeline* p, int iteration, const uint8_t** obs, const int32_t** actions, const float** rewards,
                        const uint8_t** dones, const float** behaviour_logits, const float** values, const float** stats);
/* Host arithmetic: the policy version the actor uses for rollout `iteration` (from 1): Synchronous i; Cleanba 1, 1, 2, 3, ... */
int cb_pipeline_policy_version(int sync, int iteration);
/* The synthetic environment by itself (tests): state int32 [B, cb_env_state_ints()], obs uint8 [B,C,H,W]; step reads obs_in and
 * writes obs_out (different buffers), rewards fp32 [B], dones uint8 [B]; global_step keys every random draw. */
size_t cb_env_state_ints(void);
int cb_env_reset(uint64_t seed, int B, int C, int H, int W, int32_t* state, uint8_t* obs, void* stream);
int cb_env_step(uint64_t seed, int B, int C, int H, int W, uint32_t global_step, const int32_t* actions, int32_t* state,
                const uint8_t* obs_in, uint8_t* obs_out, float* rewards, uint8_t* dones, void* stream);

/* ---- instrumentation (used by bench.py; not on the product path) --------------------------- */
/* Number of kernels this library has launched in this process so far. */
uint64_t cb_launch_count(void);
/* Per-kernel-class device timing with CUDA events recorded on the launching stream around every
 * launch of a class.  cb_profile_begin(only_class): start recording; only_class < 0 = all classes,
 * otherwise only that class (two events per launch of it, nothing else changes).
 * cb_profile_end: synchronises the device, stops recording and writes up to `max` entries (classes
 * with at least one launch): returns the number written.  flops = useful 2*MAC of the launches,
 * bytes = algorithmic bytes (operands read once + results written once). */
typedef struct {
  int cls;
  char name[28];
  uint64_t launches;
  double ms, flops, bytes;
} cb_prof_entry;
int cb_profile_begin(int only_class);
int cb_profile_end(cb_prof_entry* out, int max);

/* A22: global-norm clip + RMSprop: nu <- decay nu + (1-decay) g^2; theta <- theta - lr g / sqrt(nu + eps).  Same buffer rules
 * and scratch as cb_clip_adam. */
int cb_clip_rmsprop(size_t P, float* params, float* nu, const float* grad, float lr, float decay, float eps, float max_norm,
                    float* grad_norm, void* scratch, void* stream);
/* Linear decay of the learning rate to 0 over `total` updates (Tables 2-3): lr0 (1 - min(k,total)/total).
 * Host arithmetic: the caller passes the result as cb_hparams.lr of update k. */
float cb_linear_lr(float lr0, uint64_t k, uint64_t total);

const char* cb_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* CLEANBA_H_ */
