// Internal declarations of the Cleanba hot-path library (not part of the C ABI).
// Layouts inside the library: activations NHWC ([frame, y, x, channel], channel fastest) in the
// mode's storage type (fp32 in CB_PREC_FP32_REF, bf16 in CB_PREC_BF16_TC); every linear layer
// (conv, fc, heads) is a convolution: fc = a VALID conv whose kernel covers the whole feature map,
// heads = a 1x1 conv with A+1 outputs (A logits, then the value).
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>
#include <stddef.h>
#include <algorithm>
#include <cstring>
#include <utility>
#include <cmath>
#include <string>
#include <vector>

#include "../../include/cleanba.h"

namespace cb {

typedef __nv_bfloat16 bf16;

// one convolution-shaped linear layer
struct Geom {
  int H, W, Cin;       // input map
  int Ho, Wo, Cout;    // output map
  int kh, kw, s, p;    // kernel, stride, zero padding (low side = high side)
};

// where the layer's parameters live in the canonical flat fp32 buffer.  Output channels
// n < n_split use (w_off, b_off); the others (w2_off, b2_off) -- only the heads layer splits
// (pi.w/pi.b then v.w/v.b).
struct ParamMap {
  size_t w_off, b_off, w2_off, b2_off;
  int n_split;
  __host__ __device__ size_t w(int n, int c, int di, int dj, const Geom& g) const {
    return n < n_split ? w_off + (((size_t)n * g.Cin + c) * g.kh + di) * g.kw + dj
                       : w2_off + (((size_t)(n - n_split) * g.Cin + c) * g.kh + di) * g.kw + dj;
  }
  __host__ __device__ size_t b(int n) const { return n < n_split ? b_off + n : b2_off + (n - n_split); }
};

struct Layer {
  Geom g;
  ParamMap pm;
  int in_t, out_t, skip_t;   // activation tensor ids (-1 = observations / none)
  bool relu_in;              // the layer applies ReLU to its input when loading it
  bool gate_in;              // the input reaches the layer through a ReLU (applied here or stored by the producer): its sign gates dgrad
  bool relu_out;             // the layer stores relu(output): every consumer reads it through a ReLU anyway (first conv of a residual block)
  bool u8_in;                // first layer: uint8 NCHW observations, scaled by 1/255 (O1)
  bool f32_out;              // heads: fp32 output in every mode
  size_t wf_off, wd_off, bias_off;   // offsets (elements) into the packed weight / bias buffers
  std::string name;
};

enum OpKind { OP_CONV, OP_POOL, OP_WGRAD, OP_DGRAD, OP_POOLBWD };
enum GradBuf { G_NONE = -1, G_HEAD = 0, G_HID, G_A, G_B, G_C, G_COUNT };

struct Op {
  OpKind kind;
  int layer;        // CONV / WGRAD / DGRAD
  int in_t, out_t;  // POOL fwd: tensors;  POOLBWD: in_t = conv-output tensor (pool input)
  int C, H, W;      // POOL geometry (input map)
  int dy, dx;       // backward: gradient buffers (GradBuf)
  int mask_t;       // DGRAD: tensor whose sign gates the result (-1 none); POOL / POOLBWD: uint8 arg-max tensor
  int add;          // DGRAD: gradient buffer added after masking (-1 none)
};

// one entry per layer of the single-launch weight-packing kernel
struct PackDesc { Geom g; ParamMap pm; size_t wf_off, bias_off; int tc, conv0, dense; };

struct Tensor { size_t per_frame; bool f32; int esize; };   // esize: bytes per element, 0 = the mode's storage type

struct Workspace {     // one per precision mode
  int frames = 0;
  std::vector<void*> act;            // per tensor, [frames * per_frame]
  void* grad[G_COUNT] = {nullptr, nullptr, nullptr, nullptr, nullptr};
  void* wf = nullptr; void* wd = nullptr; float* bias = nullptr;   // packed weights (mode type), fp32 bias
  bool packed = false;                                             // the packs hold the params of the last pack_weights call
  bf16* w0img = nullptr;                                           // first-layer forward B image (conv0_tc.cu)
  bf16* wtc_f = nullptr; bf16* wtc_d = nullptr;                     // tcgen05 B-operand packs (forward / dgrad), bf16 mode only
  PackDesc* packtab = nullptr;                                     // device copy of the layer table for packing
  int* errflag = nullptr;                                          // device word, set by a kernel whose tcgen05 pipeline timed out
  int* errhost = nullptr;                                          // mapped pinned host word: set by the step's last kernel when errflag is
  float* partial = nullptr; size_t partial_elems = 0;             // wgrad split-K partials
  float* partial_tc = nullptr; size_t partial_tc_elems = 0;       // one slot per tensor-core 3x3 layer: their reductions run as ONE launch after the backward pass
  float* gradbuf = nullptr;          // [P]
  // learner scratch (fp32 unless noted)
  float *logpi = nullptr, *logmu = nullptr, *ent = nullptr, *t0 = nullptr, *t1 = nullptr, *rho = nullptr, *values = nullptr;
  float* terms = nullptr;            // (unused since the loss kernels sum their terms per block)
  double* red = nullptr;             // [0..1] advantage mean / std; [8..] per-block partial sums of the five loss terms
  float* advstat = nullptr;          // [2] mean, 1/(std+eps)
  int32_t* perm = nullptr;           // [epochs, N]  (IMPALA env groups: frame indices [(T+1) * B/mb])
  int32_t* act_m = nullptr; float* rew_m = nullptr; uint8_t* dones_m = nullptr; float* logmu_m = nullptr;   // env-group copies [T, B/mb]
  uint32_t* permj = nullptr;
  void* adam_scratch = nullptr;
  float* gnorm = nullptr;
  int learn_frames = 0; int learn_N = 0; int learn_epochs = 0;
};

}  // namespace cb

struct cb_net {
  cb_arch arch;
  int max_frames;
  size_t P;
  std::vector<cb::Layer> layers;
  std::vector<cb::Tensor> tensors;
  std::vector<cb::Op> fwd, bwd;
  size_t grad_elems[cb::G_COUNT];      // per frame
  size_t wf_total, wd_total, bias_total, partial_max;
  int head_t, hid_t;
  struct PT { std::string name; size_t off; int rank; int dims[4]; int fan_in; };
  std::vector<PT> ptensors;
  cb::Workspace ws[2];
  int last_prec = -1; int last_F = 0, last_N = 0; bool last_ppo = false; bool last_has_head = true;
  // context of a learner call in progress (cb_learner_begin .. last cb_learner_apply)
  struct LearnCtx {
    bool active = false; int n_updates = 0, next_grad = 0, next_apply = 0;
    float *params = nullptr, *adam_m = nullptr, *adam_v = nullptr; uint64_t* opt_step = nullptr;
    const uint8_t* obs = nullptr; const int32_t* actions = nullptr; const float* rewards = nullptr; const uint8_t* dones = nullptr;
    float* stats = nullptr; cb_hparams hp; int mb = 1; bool ppo = false;
  } lc;
  // actor side: the trunk of cb_policy_forward replayed as a CUDA graph per (precision, B, obs pointer); see api.cu
  struct FwdGraph { int prec, B; const uint8_t* obs; cudaGraphExec_t exec; uint64_t launches; bool bad; };
  std::vector<FwdGraph> fwd_graphs;
  cudaStream_t capture_stream = nullptr;
  cudaStream_t aux_stream = nullptr; cudaEvent_t ev_fork = nullptr, ev_join = nullptr;      // side stream of the learner (PPO permutations)
};

namespace cb {

void set_error(const char* fmt, ...);
int cuda_fail(cudaError_t e, const char* what);
#define CB_CUDA(x) do { cudaError_t e__ = (x); if (e__ != cudaSuccess) return cb::cuda_fail(e__, #x); } while (0)

// prof.cu -- launch counter and per-class event timing
enum KClass { K_PACK = 0, K_CONV_FWD, K_POOL_FWD, K_CONV_DGRAD, K_CONV_WGRAD, K_WGRAD_REDUCE, K_POOL_BWD, K_HEAD_MISC, K_LOGPROB,
              K_SCAN, K_LOSS, K_STATS, K_PERM, K_SQNORM, K_ADAM, K_SAMPLE, K_ENV, K_COUNT };
bool prof_active();                    // cb_profile_begin .. cb_profile_end
void prof_add_launches(uint64_t n);    // launches replayed by a CUDA graph
struct ProfScope {      // counts `n` launches of class `cls`; records an event pair around them when profiling
  ProfScope(int cls, cudaStream_t st, int n = 1, double flops = 0.0, double bytes = 0.0);
  ~ProfScope();
  int slot; cudaStream_t st;
};

// net.cu
int ensure_workspace(cb_net* net, int prec, int frames);
int ensure_learner_scratch(cb_net* net, int prec, int F, int N, int epochs);
int pack_weights(cb_net* net, int prec, const float* params, cudaStream_t st);
// taken / n_taken / logp_taken: the heads kernel also writes log pi(taken[n]) for frames n < n_taken (learner side; nullable)
int forward(cb_net* net, int prec, const uint8_t* obs, const int32_t* frame_idx, int F, cudaStream_t st, bool skip_heads = false,
            const int32_t* taken = nullptr, int n_taken = 0, float* logp_taken = nullptr);
int backward(cb_net* net, int prec, const uint8_t* obs, const int32_t* frame_idx, int F, float* grad, cudaStream_t st);

// conv_tc.cu
bool conv_tc_supported(const Geom& g);
bool conv_tc_fits(int H, int W, int cin, int cout);
int launch_conv_tc(int mode, int F, int H, int W, int cin, int cout, const bf16* in, const bf16* w, const float* bias, const bf16* aux0,
                   const bf16* aux1, bf16* out, bool relu_in, bool relu_out, int* error_flag, cudaStream_t st);

// conv_pool_tc.cu: stage conv + the max-pool that follows it in one kernel (forward)
bool conv_pool_tc_supported(const Geom& g);
int launch_conv_pool_tc(const Geom& g, int F, const bf16* in, const bf16* w, const float* bias, bf16* pool_out, uint8_t* pool_arg, int* error_flag, cudaStream_t st);

// wgrad_tc.cu
bool wgrad_tc_supported(const Geom& g);
size_t wgrad_tc_partial_elems(const Geom& g);
// the per-CTA partials of several layers, reduced by one launch (same fixed association per element as a per-layer launch)
struct WgradReduceJob { const float* partial; int nctas, cin_k, c_off, first_block; Geom g; ParamMap pm; };
constexpr int WGRAD_MAX_JOBS = 24;
struct WgradReduceBatch { WgradReduceJob job[WGRAD_MAX_JOBS]; int n = 0, blocks = 0; };
// `defer` != nullptr: a layer whose kernel wrote `partial` may append its reduction to the batch instead of launching it (the caller
// then gives every layer its own `partial` and calls launch_wgrad_reduce_batch before the gradient is read)
int launch_wgrad_tc(const Geom& g, const ParamMap& pm, int F, const bf16* x, const bf16* dy, bool relu_in, float* partial, float* grad,
                    int* error_flag, cudaStream_t st, WgradReduceBatch* defer = nullptr);
int launch_wgrad_reduce_batch(const WgradReduceBatch& b, float* grad, cudaStream_t st);

// conv0_tc.cu
bool conv0_tc_supported(const Geom& g);
size_t conv0_partial_elems(const Geom& g);
size_t conv0_wimg_elems(const Geom& g);
int launch_conv0_pack(const Geom& g, const ParamMap& pm, const float* params, bf16* wimg, cudaStream_t st);
int launch_conv0_fwd(const Geom& g, int F, const uint8_t* obs, const int32_t* frame_idx, const bf16* wimg, const float* bias, bf16* out,
                     bf16* pool_out, uint8_t* pool_arg, int* error_flag, cudaStream_t st);
int launch_conv0_wgrad(const Geom& g, const ParamMap& pm, int F, const uint8_t* obs, const int32_t* frame_idx, const bf16* dy, const uint8_t* pool_arg,
                       const bf16* dpool, float* partial, float* grad, int* error_flag, cudaStream_t st);

// dense_tc.cu
bool dense_tc_supported(const Geom& g);
size_t dense_partial_elems(const Geom& g, long long frames);
// wt = weight pack [N][K] (K-major, k in (y, x, c) order), wf = the SIMT forward pack [K][N]; the feature map is read as stored (the layer's
// relu_in must be false: its producer stores through the ReLU)
int launch_dense_fwd_tc(const Geom& g, int F, const bf16* A, const bf16* wt, const float* bias, bf16* out, float* partial, int* error_flag, cudaStream_t st);
int launch_dense_dgrad_tc(const Geom& g, int F, const bf16* dy, const bf16* wf, const bf16* mask, bf16* dx, int* error_flag, cudaStream_t st);
int launch_dense_wgrad_tc(const Geom& g, const ParamMap& pm, int F, const bf16* A, const bf16* dy, float* grad, int* error_flag, cudaStream_t st);

// rl.cu
int launch_sample(const float* logits, int ld, int B, int A, uint64_t seed, uint64_t step, uint32_t env_offset,
                  int32_t* actions, cudaStream_t st);
int launch_heads_sample(int prec, const void* hid, const void* wf, const float* bias, int B, int fc, int A, uint64_t seed, uint64_t step,
                        uint32_t env_offset, float* head, float* logits, float* value, int32_t* actions, cudaStream_t st,
                        const int* errflag = nullptr, int* errhost = nullptr, const int32_t* taken = nullptr, int n_taken = 0, float* logp_taken = nullptr);
int launch_split_head(const float* head, int F, int A, float* logits, float* value, cudaStream_t st);
int launch_logprob(const float* logits, int ld, int N, int A, const int32_t* actions, const int32_t* idx,
                   float* logp_a, float* entropy, cudaStream_t st);
int launch_vtrace(int T, int B, const float* V, int ldV, const float* r, const uint8_t* d, const float* logpi,
                  const float* logmu, float gamma, float lam, float rho_bar, float c_bar, float rho_pg_bar,
                  float* vs, float* pgadv, float* rho, cudaStream_t st);
int launch_gae(int T, int B, const float* V, int ldV, const float* r, const uint8_t* d, float gamma, float lam,
               float* adv, float* ret, cudaStream_t st);
int launch_permutation(uint64_t seed, uint32_t epoch0, int n_epochs, int N, int32_t* perm, uint32_t* jbuf, cudaStream_t st);
int launch_sum_ranks(const float* in, int G, size_t n, float scale, float* out, cudaStream_t st);
// env.cu
int launch_env_reset(uint64_t seed, int B, int C, int H, int W, int32_t* state, uint8_t* obs, cudaStream_t st);
int launch_env_step(uint64_t seed, int B, int C, int H, int W, uint32_t g, const int32_t* actions, int32_t* state, const uint8_t* obs_in, uint8_t* out0,
                    uint8_t* out1, float* rewards, uint8_t* dones, cudaStream_t st);
// Launch with the programmatic-stream-serialization attribute: the kernel MUST call ptx::pdl_wait() before it touches memory written by
// earlier work (tc_ptx.cuh).  Hides the launch gap and the prologue of the persistent tensor-core kernels behind the tail of their predecessor.
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
  cudaLaunchConfig_t cfg; memset(&cfg, 0, sizeof cfg);
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization; attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}
// one opt-in per (device, kernel): cudaFuncAttributeMaxDynamicSharedMemorySize raised to at least `bytes`
int ensure_dyn_smem(const void* func, size_t bytes);
// loss kernels write dhead [N, A+1] in the mode's storage type and per-sample terms; reduce writes stats
int launch_impala_loss(int prec, int N, int A, const float* head, const int32_t* act, const float* vs, const float* pgadv,
                       const float* rho, float c1, float c2, int reduction, void* dhead, float* terms, double* red,
                       float* stats, cudaStream_t st);
int launch_ppo_loss(int prec, int m, int A, const float* head, const int32_t* idx, const int32_t* act, const float* adv,
                    const float* ret, const float* logp_old, float eps, float c1, float c2, int norm_adv, void* dhead,
                    float* terms, double* red, float* advstat, float* stats, cudaStream_t st);
int launch_clip_rmsprop(size_t P, float* params, float* nu, const float* g, float lr, float decay, float eps, float max_norm, float* grad_norm,
                        float* stats_slot, void* scratch, cudaStream_t st, const int* errflag = nullptr, int* errhost = nullptr);
int launch_gather_traj(int T, int B, int b0, int Bm, const int32_t* act, const float* rew, const uint8_t* dones, const float* logmu, int32_t* fidx,
                       int32_t* act_m, float* rew_m, uint8_t* dones_m, float* logmu_m, cudaStream_t st);
size_t clip_adam_scratch_bytes(size_t P);
int launch_clip_adam(size_t P, float* params, float* m, float* v, const float* g, uint64_t k, float lr, float b1, float b2,
                     float eps, float max_norm, float* grad_norm, float* stats_slot, void* scratch, cudaStream_t st,
                     const int* errflag = nullptr, int* errhost = nullptr);

}  // namespace cb
