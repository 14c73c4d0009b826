// RL side of the hot path: distribution math and Gumbel-max sampling,
// V-trace / GAE reverse scans (a6-a7), IMPALA / PPO losses with their adjoint seeds (a8),
// the PPO permutation (a12) and global-norm clip + Adam (a11).  All reductions have a fixed order.
#include "common.cuh"

namespace cb {

constexpr int MAX_A = 32;      // n_actions + 1 must not exceed this

// ------------------------------------------------------------------------------------------------
// A9: Philox4x32-10 counter-based generator (Salmon et al. 2011), 10 rounds.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t out[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// A9: natural log as a FIXED sequence of IEEE binary64 operations, written with the _rn intrinsics
// so that the compiler can neither contract nor reorder them:  x = m 2^e, m in (sqrt(1/2), sqrt(2)];
// s = (m-1)/(m+1); log m = s * sum_k c_k s^(2k), c_k = 2/(2k+1), k = 0..12 (Horner, fma);
// log x = fma(e, LN2_HI, fma(e, LN2_LO, log m)).
__device__ __forceinline__ double fixed_log(double x) {
  const double LN2_HI = 0x1.62e42fee00000p-1, LN2_LO = 0x1.a39ef35793c76p-33, SQRT2 = 0x1.6a09e667f3bcdp+0;
  long long bits = __double_as_longlong(x);
  int e = (int)((bits >> 52) & 0x7ff) - 1023;
  double m = __longlong_as_double((bits & 0x000fffffffffffffLL) | 0x3ff0000000000000LL);
  if (m > SQRT2) { m = __dmul_rn(m, 0.5); e += 1; }
  double s = __ddiv_rn(__dadd_rn(m, -1.0), __dadd_rn(m, 1.0));
  double z = __dmul_rn(s, s);
  double p = 2.0 / 25.0;
  p = __fma_rn(p, z, 2.0 / 23.0); p = __fma_rn(p, z, 2.0 / 21.0); p = __fma_rn(p, z, 2.0 / 19.0);
  p = __fma_rn(p, z, 2.0 / 17.0); p = __fma_rn(p, z, 2.0 / 15.0); p = __fma_rn(p, z, 2.0 / 13.0);
  p = __fma_rn(p, z, 2.0 / 11.0); p = __fma_rn(p, z, 2.0 / 9.0);  p = __fma_rn(p, z, 2.0 / 7.0);
  p = __fma_rn(p, z, 2.0 / 5.0);  p = __fma_rn(p, z, 2.0 / 3.0);  p = __fma_rn(p, z, 2.0);
  double lm = __dmul_rn(s, p);
  double ed = (double)e;
  return __fma_rn(ed, LN2_HI, __fma_rn(ed, LN2_LO, lm));
}

// u = ((x >> 8) + 0.5) 2^-24 in (0,1) (exact); g = -log(-log u), rounded once to fp32
__device__ __forceinline__ float gumbel_from_u32(uint32_t x) {
  double u = __dmul_rn(__dadd_rn((double)(x >> 8), 0.5), 0x1p-24);
  double g = -fixed_log(-fixed_log(u));
  return __double2float_rn(g);
}

// O3: a = argmax_i (logit_i + g_i) in fp32, lowest index on ties; one thread per env.
__global__ void sample_kernel(const float* __restrict__ logits, int ld, int B, int A, uint32_t k0, uint32_t k1,
                              uint32_t step_lo, uint32_t step_hi, uint32_t env_offset, int32_t* __restrict__ actions) {
  int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= B) return;
  const float* l = logits + (size_t)b * ld;
  int best = 0; float bs = 0.f;
  for (int j = 0; j * 4 < A; ++j) {
    uint32_t r[4];
    philox4x32_10(env_offset + (uint32_t)b, step_lo, step_hi, (uint32_t)j, k0, k1, r);
    for (int w = 0; w < 4 && 4 * j + w < A; ++w) {
      int i = 4 * j + w;
      float sc = __fadd_rn(l[i], gumbel_from_u32(r[w]));
      if (i == 0 || sc > bs) { bs = sc; best = i; }
    }
  }
  actions[b] = best;
}

int launch_sample(const float* logits, int ld, int B, int A, uint64_t seed, uint64_t step, uint32_t env_offset, int32_t* actions, cudaStream_t st) {
  if (B <= 0) return CB_OK;
  ProfScope ps(K_SAMPLE, st);
  sample_kernel<<<(B + 63) / 64, 64, 0, st>>>(logits, ld, B, A, (uint32_t)seed, (uint32_t)(seed >> 32), (uint32_t)step, (uint32_t)(step >> 32), env_offset, actions);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

// Actor-side head epilogue in ONE kernel: one warp per env computes the A logits and the value
// from relu(hidden) (lanes stride over the hidden units, fixed shuffle tree), writes them, and draws the action:
// lane i < A forms logit_i + Gumbel_i, the warp takes the arg-max with the lowest index on ties (O3 / A9).
template <typename AT>
__global__ void heads_sample_kernel(const AT* __restrict__ hid, const AT* __restrict__ wf, const float* __restrict__ bias, int B, int fc, int A,
                                    uint32_t k0, uint32_t k1, uint32_t step_lo, uint32_t step_hi, uint32_t env_offset,
                                    float* __restrict__ head, float* __restrict__ logits, float* __restrict__ value, int32_t* __restrict__ actions,
                                    const int* __restrict__ errflag, int* errhost, const int32_t* __restrict__ taken, int n_taken, float* __restrict__ logp_taken) {
  const int b = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (b >= B) return;
  const int N = A + 1;
  if (errflag && *errflag) {      // a tcgen05 pipeline of the trunk timed out: poison the outputs, tell the host (cleanba.h, asynchronous errors)
    if (lane < N) {
      if (head) head[(size_t)b * N + lane] = NAN;
      if (lane < A) { if (logits) logits[(size_t)b * A + lane] = NAN; } else if (value) value[b] = NAN;
    }
    if (lane == 0 && actions) actions[b] = -1;
    if (b == 0 && lane == 0 && errhost) *errhost = *errflag;
    return;
  }
  float acc[MAX_A];
#pragma unroll
  for (int n = 0; n < MAX_A; ++n) acc[n] = 0.f;
  for (int k = lane; k < fc; k += 32) {
    float h;
    if (sizeof(AT) == 2) h = __bfloat162float(reinterpret_cast<const bf16*>(hid)[(size_t)b * fc + k]); else h = reinterpret_cast<const float*>(hid)[(size_t)b * fc + k];
    h = fmaxf(h, 0.f);
#pragma unroll
    for (int n = 0; n < MAX_A; ++n) if (n < N) {
      float w;
      if (sizeof(AT) == 2) w = __bfloat162float(reinterpret_cast<const bf16*>(wf)[(size_t)k * N + n]); else w = reinterpret_cast<const float*>(wf)[(size_t)k * N + n];
      acc[n] = fmaf(h, w, acc[n]);
    }
  }
  float mine = 0.f;      // lane n ends up holding output n
#pragma unroll
  for (int n = 0; n < MAX_A; ++n) if (n < N) {
    float v = acc[n];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (lane == n) mine = v + bias[n];
  }
  if (lane < N) {
    if (head) head[(size_t)b * N + lane] = mine;
    if (lane < A) { if (logits) logits[(size_t)b * A + lane] = mine; } else if (value) value[b] = mine;
  }
  if (logp_taken && b < n_taken) {
    // learner side (a4): log pi(a_t | s_t) of the action the rollout took, from the warp's own logits: lse = max + log sum exp(l - max)
    // in fp64 with a fixed xor-shuffle tree (the arithmetic of logprob_kernel, without a second pass over the logits)
    const double l = lane < A ? (double)mine : -INFINITY;
    double m = l;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    double s = lane < A ? exp(l - m) : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    const int a = min(max(taken[b], 0), A - 1);
    const double la = __shfl_sync(0xffffffffu, l, a);
    if (lane == 0) logp_taken[b] = (float)(la - (m + log(s)));
  }
  if (actions) {
    float sc = -INFINITY;
    if (lane < A) {
      uint32_t r[4];
      philox4x32_10(env_offset + (uint32_t)b, step_lo, step_hi, (uint32_t)(lane >> 2), k0, k1, r);
      sc = __fadd_rn(mine, gumbel_from_u32(r[lane & 3]));
    }
    int best = lane;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      float os = __shfl_xor_sync(0xffffffffu, sc, o); int ob = __shfl_xor_sync(0xffffffffu, best, o);
      if (os > sc || (os == sc && ob < best)) { sc = os; best = ob; }
    }
    if (lane == 0) actions[b] = best;
  }
}

int launch_heads_sample(int prec, const void* hid, const void* wf, const float* bias, int B, int fc, int A, uint64_t seed, uint64_t step,
                        uint32_t env_offset, float* head, float* logits, float* value, int32_t* actions, cudaStream_t st,
                        const int* errflag, int* errhost, const int32_t* taken, int n_taken, float* logp_taken) {
  if (B <= 0) return CB_OK;
  if (A + 1 > MAX_A) { set_error("n_actions too large"); return CB_EINVAL; }
  ProfScope ps(K_SAMPLE, st);
  const int grid = (B * 32 + 127) / 128;
  if (prec == CB_PREC_FP32_REF)
    heads_sample_kernel<float><<<grid, 128, 0, st>>>((const float*)hid, (const float*)wf, bias, B, fc, A, (uint32_t)seed, (uint32_t)(seed >> 32), (uint32_t)step,
                                                      (uint32_t)(step >> 32), env_offset, head, logits, value, actions, errflag, errhost, taken, n_taken, logp_taken);
  else
    heads_sample_kernel<bf16><<<grid, 128, 0, st>>>((const bf16*)hid, (const bf16*)wf, bias, B, fc, A, (uint32_t)seed, (uint32_t)(seed >> 32), (uint32_t)step,
                                                     (uint32_t)(step >> 32), env_offset, head, logits, value, actions, errflag, errhost, taken, n_taken, logp_taken);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

__global__ void split_head_kernel(const float* __restrict__ head, int F, int A, float* __restrict__ logits, float* __restrict__ value) {
  size_t total = (size_t)F * (A + 1);
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    size_t f = i / (A + 1); int a = (int)(i - f * (A + 1));
    if (a < A) { if (logits) logits[f * A + a] = head[i]; } else if (value) value[f] = head[i];
  }
}
int launch_split_head(const float* head, int F, int A, float* logits, float* value, cudaStream_t st) {
  size_t total = (size_t)F * (A + 1); if (!total) return CB_OK;
  ProfScope ps(K_HEAD_MISC, st);
  split_head_kernel<<<(int)std::min<size_t>((total + 255) / 256, 2368), 256, 0, st>>>(head, F, A, logits, value);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

// ------------------------------------------------------------------------------------------------
// O2: lse = max + log sum exp(l - max); log p = l - lse; H = -sum p log p.   R = compute type.
// ------------------------------------------------------------------------------------------------
template <typename R> __device__ __forceinline__ R rexp(R x);
template <> __device__ __forceinline__ float rexp<float>(float x) { return expf(x); }
template <> __device__ __forceinline__ double rexp<double>(double x) { return exp(x); }
template <typename R> __device__ __forceinline__ R rlog(R x);
template <> __device__ __forceinline__ float rlog<float>(float x) { return logf(x); }
template <> __device__ __forceinline__ double rlog<double>(double x) { return log(x); }


// lse and entropy of one row without a per-thread array (a runtime-indexed array would live in local memory): log p_i = l_i - lse is
// recomputed where it is needed.
template <typename R>
__device__ __forceinline__ void lse_entropy(const float* l, int A, R* lse_out, R* H) {
  R m = (R)l[0];
  for (int i = 1; i < A; ++i) m = max(m, (R)l[i]);
  R s = 0;
  for (int i = 0; i < A; ++i) s += rexp<R>((R)l[i] - m);
  const R lse = m + rlog<R>(s);
  R h = 0;
  for (int i = 0; i < A; ++i) { const R lp = (R)l[i] - lse; h -= rexp<R>(lp) * lp; }
  *lse_out = lse; *H = h;
}

// Rows of `ld` floats (A logits first) for ROWS consecutive samples are contiguous in global memory: the block copies them to shared
// memory with coalesced loads (row pitch ld + (ld even): odd, so that a thread walking its own row does not collide with its
// neighbours' banks), one thread then owns one sample.
constexpr int LP_ROWS = 128;
__device__ __forceinline__ int lp_pitch(int ld) { return ld | 1; }
__device__ __forceinline__ void stage_rows(const float* __restrict__ g, int ld, int n0, int nrows, float* sh) {
  const int tot = nrows * ld, pitch = lp_pitch(ld);
  const float* src = g + (size_t)n0 * ld;
  const int dr = (int)blockDim.x / ld, dc = (int)blockDim.x - dr * ld;      // (row, column) advance per pass: no division in the loop
  int r = (int)threadIdx.x / ld, c = (int)threadIdx.x - r * ld;
  for (int i = threadIdx.x; i < tot; i += blockDim.x) {
    sh[r * pitch + c] = src[i];
    r += dr; c += dc; if (c >= ld) { c -= ld; ++r; }
  }
}

__global__ void __launch_bounds__(LP_ROWS) logprob_kernel(const float* __restrict__ logits, int ld, int N, int A, const int32_t* __restrict__ actions,
                                                          const int32_t* __restrict__ idx, float* __restrict__ logp_a, float* __restrict__ entropy) {
  extern __shared__ float lp_sh[];
  const int n0 = blockIdx.x * LP_ROWS, nrows = min(LP_ROWS, N - n0), n = n0 + threadIdx.x;
  stage_rows(logits, ld, n0, nrows, lp_sh);
  __syncthreads();
  if (n >= N) return;
  const float* l = lp_sh + threadIdx.x * lp_pitch(ld);
  double lse, H;
  lse_entropy<double>(l, A, &lse, &H);
  int a = min(max(actions[idx ? idx[n] : n], 0), A - 1);      // never index out of bounds with a bad action (cleanba.h)
  if (logp_a) logp_a[n] = (float)((double)l[a] - lse);
  if (entropy) entropy[n] = (float)H;
}
int launch_logprob(const float* logits, int ld, int N, int A, const int32_t* actions, const int32_t* idx, float* logp_a, float* entropy, cudaStream_t st) {
  if (N <= 0) return CB_OK;
  if (ld > 64) { set_error("logprob: row length > 64"); return CB_EINVAL; }
  ProfScope ps(K_LOGPROB, st, 1, 0.0, (double)N * (ld * 4.0 + 4 + (logp_a ? 4 : 0) + (entropy ? 4 : 0)));
  logprob_kernel<<<(N + LP_ROWS - 1) / LP_ROWS, LP_ROWS, (size_t)LP_ROWS * (ld | 1) * 4, st>>>(logits, ld, N, A, actions, idx, logp_a, entropy);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

// ------------------------------------------------------------------------------------------------
// O4 V-trace (A2) and O6 GAE (A3): one lane per env, t = T-1 .. 0; adjacent lanes read adjacent
// envs of a [T,B] row, so every access is coalesced and the operation order is the definition's.
// ------------------------------------------------------------------------------------------------
__global__ void vtrace_kernel(int T, int B, const float* __restrict__ V, int ldV, const float* __restrict__ r, const uint8_t* __restrict__ d,
                              const float* __restrict__ logpi, const float* __restrict__ logmu, float gamma, float lam, float rho_bar,
                              float c_bar, float rho_pg_bar, float* __restrict__ vs, float* __restrict__ pgadv, float* __restrict__ rho_out) {
  int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= B) return;
  float Vn = V[((size_t)T * B + b) * ldV];
  float acc = 0.f, vs_next = Vn;
#pragma unroll 8
  for (int t = T - 1; t >= 0; --t) {      // loads of eight steps in flight; the recurrence runs in the definition's order
    size_t i = (size_t)t * B + b;
    float Vt = V[i * ldV];
    float disc = gamma * (1.0f - (float)d[i]);
    float w = expf(logpi[i] - logmu[i]);
    float rho = fminf(rho_bar, w), c = lam * fminf(c_bar, w);
    float delta = rho * (r[i] + disc * Vn - Vt);
    acc = delta + disc * c * acc;
    float q = r[i] + disc * (lam * vs_next + (1.0f - lam) * Vn);
    pgadv[i] = fminf(rho_pg_bar, w) * (q - Vt);
    float v = Vt + acc;
    vs[i] = v; vs_next = v; Vn = Vt;
    if (rho_out) rho_out[i] = rho;
  }
}
int launch_vtrace(int T, int B, const float* V, int ldV, const float* r, const uint8_t* d, const float* logpi, const float* logmu,
                  float gamma, float lam, float rho_bar, float c_bar, float rho_pg_bar, float* vs, float* pgadv, float* rho, cudaStream_t st) {
  if (B <= 0 || T <= 0) return CB_OK;
  ProfScope ps(K_SCAN, st, 1, 0.0, (double)T * B * (4 * 4 + 1 + 3 * 4) + B * 4.0);
  vtrace_kernel<<<(B + 127) / 128, 128, 0, st>>>(T, B, V, ldV, r, d, logpi, logmu, gamma, lam, rho_bar, c_bar, rho_pg_bar, vs, pgadv, rho);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

__global__ void gae_kernel(int T, int B, const float* __restrict__ V, int ldV, const float* __restrict__ r, const uint8_t* __restrict__ d,
                           float gamma, float lam, float* __restrict__ adv, float* __restrict__ ret) {
  int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= B) return;
  float Vn = V[((size_t)T * B + b) * ldV], a = 0.f;
#pragma unroll 8
  for (int t = T - 1; t >= 0; --t) {      // loads of eight steps in flight; the recurrence runs in the definition's order
    size_t i = (size_t)t * B + b;
    float Vt = V[i * ldV];
    float disc = gamma * (1.0f - (float)d[i]);
    float delta = r[i] + disc * Vn - Vt;
    a = delta + disc * lam * a;
    adv[i] = a; ret[i] = a + Vt; Vn = Vt;
  }
}
int launch_gae(int T, int B, const float* V, int ldV, const float* r, const uint8_t* d, float gamma, float lam, float* adv, float* ret, cudaStream_t st) {
  if (B <= 0 || T <= 0) return CB_OK;
  ProfScope ps(K_SCAN, st, 1, 0.0, (double)T * B * (2 * 4 + 1 + 2 * 4) + B * 4.0);
  gae_kernel<<<(B + 127) / 128, 128, 0, st>>>(T, B, V, ldV, r, d, gamma, lam, adv, ret);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

// ------------------------------------------------------------------------------------------------
// A17: per-epoch Fisher-Yates.  Draw q is word q%4 of Philox block (q/4, epoch, 0, 0x5045524D), key =
// perm_seed; for i = N-1 .. 1: j = (x_q * (i+1)) >> 32, swap(perm[i], perm[j]).  The draws are
// computed in parallel, the swaps (inherently serial) by one thread; one block per epoch.
// ------------------------------------------------------------------------------------------------
// SMEM: the index array lives in shared memory during the swap loop (one dependent shared-memory round trip per swap
// instead of an L2 round trip); N * 4 bytes must fit the opt-in limit, otherwise the loop runs on the global array.
template <bool SMEM>
__global__ void permutation_kernel(uint32_t k0, uint32_t k1, uint32_t epoch0, int N, int32_t* __restrict__ perm_all, uint32_t* __restrict__ j_all) {
  extern __shared__ int32_t sperm[];
  uint32_t epoch = epoch0 + blockIdx.x;
  int32_t* perm = perm_all + (size_t)blockIdx.x * N;
  uint32_t* jb = j_all + (size_t)blockIdx.x * N;
  for (int q4 = threadIdx.x; q4 * 4 < N - 1; q4 += blockDim.x) {
    uint32_t r[4]; philox4x32_10((uint32_t)q4, epoch, 0u, 0x5045524Du, k0, k1, r);
    for (int w = 0; w < 4; ++w) {
      int q = q4 * 4 + w; int i = N - 1 - q;
      if (i >= 1) jb[q] = (uint32_t)(((uint64_t)r[w] * (uint64_t)(i + 1)) >> 32);
    }
  }
  int32_t* wk = SMEM ? sperm : perm;
  for (int i = threadIdx.x; i < N; i += blockDim.x) wk[i] = i;
  __syncthreads();
  if (threadIdx.x == 0) {
    int i = N - 1, q = 0;
    for (; i >= 8; i -= 8, q += 8) {      // the eight draws of a pass are fetched together; the swaps stay in order
      uint32_t j[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) j[u] = jb[q + u];
#pragma unroll
      for (int u = 0; u < 8; ++u) { int32_t a = wk[i - u], b = wk[j[u]]; wk[i - u] = b; wk[j[u]] = a; }
    }
    for (; i >= 1; --i, ++q) { uint32_t j = jb[q]; int32_t a = wk[i], b = wk[j]; wk[i] = b; wk[j] = a; }
  }
  if (SMEM) {
    __syncthreads();
    for (int i = threadIdx.x; i < N; i += blockDim.x) perm[i] = sperm[i];
  }
}
int launch_permutation(uint64_t seed, uint32_t epoch0, int n_epochs, int N, int32_t* perm, uint32_t* jbuf, cudaStream_t st) {
  if (N <= 0 || n_epochs <= 0) return CB_OK;
  ProfScope ps(K_PERM, st);
  const size_t smem = (size_t)N * 4;
  if (smem <= 200 * 1024) {
    if (smem > 48 * 1024) { int rc = ensure_dyn_smem((const void*)permutation_kernel<true>, smem); if (rc) return rc; }
    permutation_kernel<true><<<n_epochs, 256, smem, st>>>((uint32_t)seed, (uint32_t)(seed >> 32), epoch0, N, perm, jbuf);
  } else
    permutation_kernel<false><<<n_epochs, 256, 0, st>>>((uint32_t)seed, (uint32_t)(seed >> 32), epoch0, N, perm, jbuf);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

// fixed-order sum over ranks (cb_sum_ranks): out[i] = scale * (in[0][i] + ... + in[G-1][i]), added in rank order
template <bool VEC>      // VEC: n % 4 == 0 and 16-byte aligned buffers, so that every rank's slice can be read as float4
__global__ void __launch_bounds__(256) sum_ranks_kernel(const float* __restrict__ in, int G, size_t n, float scale, float* __restrict__ out) {
  if (VEC) {
    const size_t nv = n / 4;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < nv; i += (size_t)gridDim.x * blockDim.x) {
      float4 s = reinterpret_cast<const float4*>(in)[i];
      for (int r = 1; r < G; ++r) { const float4 x = reinterpret_cast<const float4*>(in + (size_t)r * n)[i]; s.x += x.x; s.y += x.y; s.z += x.z; s.w += x.w; }
      s.x *= scale; s.y *= scale; s.z *= scale; s.w *= scale;
      reinterpret_cast<float4*>(out)[i] = s;
    }
  } else {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
      float s = in[i];
      for (int r = 1; r < G; ++r) s += in[(size_t)r * n + i];
      out[i] = s * scale;
    }
  }
}
int launch_sum_ranks(const float* in, int G, size_t n, float scale, float* out, cudaStream_t st) {
  if (n == 0 || G <= 0) return CB_OK;
  ProfScope ps(K_HEAD_MISC, st, 1, 0.0, (double)n * 4 * (G + 1));
  const bool vec = (n & 3) == 0 && (((uintptr_t)in | (uintptr_t)out) & 15) == 0;
  int grid = (int)std::min<size_t>(((vec ? n / 4 : n) + 255) / 256, (size_t)148 * 8); if (grid < 1) grid = 1;
  if (vec) sum_ranks_kernel<true><<<grid, 256, 0, st>>>(in, G, n, scale, out);
  else sum_ranks_kernel<false><<<grid, 256, 0, st>>>(in, G, n, scale, out);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

// ------------------------------------------------------------------------------------------------
// Fixed-order block reduction in fp64: thread-strided serial sums, then a shared-memory tree.
// ------------------------------------------------------------------------------------------------
template <int NT>
__device__ __forceinline__ double block_sum(double v, double* sh) {
  sh[threadIdx.x] = v; __syncthreads();
  for (int s = NT / 2; s > 0; s >>= 1) { if ((int)threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s]; __syncthreads(); }
  double r = sh[0]; __syncthreads();
  return r;
}

template <typename AT> __device__ __forceinline__ void st_grad(AT* p, size_t i, float v);
template <> __device__ __forceinline__ void st_grad<float>(float* p, size_t i, float v) { p[i] = v; }
template <> __device__ __forceinline__ void st_grad<bf16>(bf16* p, size_t i, float v) { p[i] = __float2bfloat16_rn(v); }

// ---- losses (a8).  One thread per sample, LP_ROWS samples per block.  The block's head rows come in through shared memory
// (coalesced), the seeds leave through shared memory (coalesced), and the five per-sample terms are summed per block in fp64 (fixed
// tree) into partial[block][5]; stats_final_kernel adds the block partials in block order.  The association is a function of N only.
template <typename AT>
__device__ __forceinline__ void store_seed_rows(AT* __restrict__ dhead, int ld, int n0, int nrows, const float* sh) {
  const int tot = nrows * ld, pitch = lp_pitch(ld);
  AT* dst = dhead + (size_t)n0 * ld;
  const int dr = (int)blockDim.x / ld, dc = (int)blockDim.x - dr * ld;
  int r = (int)threadIdx.x / ld, c = (int)threadIdx.x - r * ld;
  for (int i = threadIdx.x; i < tot; i += blockDim.x) {
    st_grad<AT>(dst, (size_t)i, sh[r * pitch + c]);
    r += dr; c += dc; if (c >= ld) { c -= ld; ++r; }
  }
}
// the five per-sample terms summed over the block in fp64: xor-shuffle tree inside each warp (a fixed association), then the warp sums
// in warp order
__device__ __forceinline__ void block_terms(double (&t)[5], double* shd, double* __restrict__ partial) {
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    double v = t[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) shd[(threadIdx.x >> 5) * 5 + k] = v;
  }
  __syncthreads();
  if (threadIdx.x < 5) {
    double s = 0.0;
    for (int w = 0; w < LP_ROWS / 32; ++w) s += shd[w * 5 + threadIdx.x];
    partial[(size_t)blockIdx.x * 5 + threadIdx.x] = s;
  }
}

// O5 IMPALA loss terms + adjoint seeds (A4-A6).  terms = pg, v, H, rho, 0.
template <typename AT, typename R>
__global__ void __launch_bounds__(LP_ROWS) impala_loss_kernel(int N, int A, const float* __restrict__ head, const int32_t* __restrict__ act, const float* __restrict__ vs,
                                                              const float* __restrict__ pgadv, const float* __restrict__ rho, float c1, float c2, float inv,
                                                              AT* __restrict__ dhead, double* __restrict__ partial) {
  extern __shared__ float lp_sh[];
  __shared__ double shd[LP_ROWS];
  const int ld = A + 1, n0 = blockIdx.x * LP_ROWS, nrows = min(LP_ROWS, N - n0), n = n0 + threadIdx.x;
  stage_rows(head, ld, n0, nrows, lp_sh);
  __syncthreads();
  double t[5] = {0, 0, 0, 0, 0};
  if (n < N) {
    float* l = lp_sh + threadIdx.x * lp_pitch(ld);
    R lse, H;
    lse_entropy<R>(l, A, &lse, &H);
    const int a = min(max(act[n], 0), A - 1);
    const R pg = (R)pgadv[n], err = (R)vs[n] - (R)l[A], lpa = (R)l[a] - lse;
    for (int i = 0; i < A; ++i) {
      const R lp = (R)l[i] - lse, p = rexp<R>(lp);
      l[i] = (float)((R)inv * (-pg * ((i == a ? (R)1 : (R)0) - p) + (R)c2 * p * (lp + H)));      // the row is overwritten by its seeds
    }
    l[A] = (float)(-(R)c1 * err * (R)inv);
    t[0] = (double)(float)(-pg * lpa); t[1] = (double)(float)((R)0.5 * err * err); t[2] = (double)(float)H; t[3] = rho ? (double)rho[n] : 0.0;
  }
  __syncthreads();
  store_seed_rows<AT>(dhead, ld, n0, nrows, lp_sh);
  block_terms(t, shd, partial);
}

// adds the block partials [nblk][5] in block order (fp64) and writes the stats record.  mode 0 IMPALA, 1 PPO.
__global__ void __launch_bounds__(256) stats_final_kernel(int N, int nblk, const double* __restrict__ partial, int mode, float c1, float c2, int reduction, float* __restrict__ stats) {
  __shared__ double sh[256];
  double s[5];
  for (int k = 0; k < 5; ++k) {
    double v = 0.0;
    for (int i = threadIdx.x; i < nblk; i += 256) v += partial[(size_t)i * 5 + k];
    s[k] = block_sum<256>(v, sh);
  }
  if (threadIdx.x == 0) {
    double invN = 1.0 / (double)N, inv = (mode == 0 && reduction == 1) ? 1.0 : invN;
    double pg = s[0] * inv, vl = s[1] * inv;
    stats[1] = (float)pg; stats[2] = (float)vl; stats[3] = (float)(s[2] * invN);
    stats[0] = (float)(pg + (double)c1 * vl - (double)c2 * (s[2] * inv));
    stats[4] = 0.f;
    stats[5] = mode == 1 ? (float)(s[3] * invN) : 0.f;
    stats[6] = mode == 1 ? (float)(s[4] * invN) : 0.f;
    stats[7] = mode == 0 ? (float)(s[3] * invN) : 0.f;
  }
}

size_t loss_partial_doubles(int N) { return (size_t)((N + LP_ROWS - 1) / LP_ROWS) * 5 + 8; }

int launch_impala_loss(int prec, int N, int A, const float* head, const int32_t* act, const float* vs, const float* pgadv, const float* rho,
                       float c1, float c2, int reduction, void* dhead, float*, double* red, float* stats, cudaStream_t st) {
  if (A + 1 > MAX_A) { set_error("n_actions > %d", MAX_A - 1); return CB_EINVAL; }
  float inv = reduction == 0 ? (float)(1.0 / (double)N) : 1.0f;
  const int grid = (N + LP_ROWS - 1) / LP_ROWS; const size_t smem = (size_t)LP_ROWS * ((A + 1) | 1) * 4;
  double* partial = red + 8;
  { ProfScope ps(K_LOSS, st, 1, 0.0, (double)N * ((A + 1) * (4.0 + (prec ? 2 : 4)) + 16));
  if (prec == CB_PREC_FP32_REF) impala_loss_kernel<float, double><<<grid, LP_ROWS, smem, st>>>(N, A, head, act, vs, pgadv, rho, c1, c2, inv, (float*)dhead, partial);
  else impala_loss_kernel<bf16, float><<<grid, LP_ROWS, smem, st>>>(N, A, head, act, vs, pgadv, rho, c1, c2, inv, (bf16*)dhead, partial); }
  ProfScope ps2(K_STATS, st, 1, 0.0, (double)grid * 40);
  stats_final_kernel<<<1, 256, 0, st>>>(N, grid, partial, 0, c1, c2, reduction, stats);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

// A8: population mean / std of the minibatch advantages, two-pass, fp64, fixed order. red[0]=mean, red[1]=std
__global__ void __launch_bounds__(1024) adv_stats_kernel(int m, const int32_t* __restrict__ idx, const float* __restrict__ adv, double* __restrict__ red) {
  __shared__ double sh[1024];
  double v = 0.0;
  for (int i = threadIdx.x; i < m; i += 1024) v += (double)adv[idx ? idx[i] : i];
  double mean = block_sum<1024>(v, sh) / (double)m;
  v = 0.0;
  for (int i = threadIdx.x; i < m; i += 1024) { double dlt = (double)adv[idx ? idx[i] : i] - mean; v += dlt * dlt; }
  double var = block_sum<1024>(v, sh) / (double)m;
  if (threadIdx.x == 0) { red[0] = mean; red[1] = sqrt(var); }
}

// O7 PPO loss terms + adjoint seeds (Eq. 2-3; A5-A8).  terms = pg, v, H, kl, clip.
template <typename AT, typename R>
__global__ void __launch_bounds__(LP_ROWS) ppo_loss_kernel(int m, int A, const float* __restrict__ head, const int32_t* __restrict__ idx, const int32_t* __restrict__ act,
                                                           const float* __restrict__ adv, const float* __restrict__ ret, const float* __restrict__ logp_old, float eps,
                                                           float c1, float c2, int norm_adv, const double* __restrict__ red, AT* __restrict__ dhead,
                                                           double* __restrict__ partial) {
  extern __shared__ float lp_sh[];
  __shared__ double shd[LP_ROWS];
  const int ld = A + 1, n0 = blockIdx.x * LP_ROWS, nrows = min(LP_ROWS, m - n0), n = n0 + threadIdx.x;
  stage_rows(head, ld, n0, nrows, lp_sh);
  __syncthreads();
  double t[5] = {0, 0, 0, 0, 0};
  if (n < m) {
    const int src = idx ? idx[n] : n;
    float* l = lp_sh + threadIdx.x * lp_pitch(ld);
    R lse, H;
    lse_entropy<R>(l, A, &lse, &H);
    const int a = min(max(act[src], 0), A - 1);
    const R inv = (R)(1.0 / (double)m);
    const R At = norm_adv ? (R)(((double)adv[src] - red[0]) / (red[1] + 1e-8)) : (R)adv[src];
    const R logr = ((R)l[a] - lse) - (R)logp_old[src], r = rexp<R>(logr);
    const R lo = (R)1 - (R)eps, hi = (R)1 + (R)eps;
    const R rc = min(max(r, lo), hi);
    const R l1 = -At * r, l2 = -At * rc;
    const bool clipped = (At > 0 && r > hi) || (At < 0 && r < lo);   // strictly clipped on the penalised side (A7)
    const R dlogp = clipped ? (R)0 : -At * r * inv;
    const R err = (R)l[A] - (R)ret[src];
    for (int i = 0; i < A; ++i) {
      const R lp = (R)l[i] - lse, p = rexp<R>(lp);
      l[i] = (float)(dlogp * ((i == a ? (R)1 : (R)0) - p) + inv * (R)c2 * p * (lp + H));
    }
    l[A] = (float)((R)c1 * err * inv);
    R ar = r - (R)1; if (ar < 0) ar = -ar;
    t[0] = (double)(float)max(l1, l2); t[1] = (double)(float)((R)0.5 * err * err); t[2] = (double)(float)H;
    t[3] = (double)(float)((r - (R)1) - logr); t[4] = ar > (R)eps ? 1.0 : 0.0;
  }
  __syncthreads();
  store_seed_rows<AT>(dhead, ld, n0, nrows, lp_sh);
  block_terms(t, shd, partial);
}

int launch_ppo_loss(int prec, int m, int A, const float* head, const int32_t* idx, const int32_t* act, const float* adv, const float* ret,
                    const float* logp_old, float eps, float c1, float c2, int norm_adv, void* dhead, float*, double* red, float*,
                    float* stats, cudaStream_t st) {
  if (A + 1 > MAX_A) { set_error("n_actions > %d", MAX_A - 1); return CB_EINVAL; }
  if (norm_adv) { ProfScope ps0(K_STATS, st); adv_stats_kernel<<<1, 1024, 0, st>>>(m, idx, adv, red); }
  const int grid = (m + LP_ROWS - 1) / LP_ROWS; const size_t smem = (size_t)LP_ROWS * ((A + 1) | 1) * 4;
  double* partial = red + 8;
  { ProfScope ps(K_LOSS, st, 1, 0.0, (double)m * ((A + 1) * (4.0 + (prec ? 2 : 4)) + 20));
  if (prec == CB_PREC_FP32_REF) ppo_loss_kernel<float, double><<<grid, LP_ROWS, smem, st>>>(m, A, head, idx, act, adv, ret, logp_old, eps, c1, c2, norm_adv, red, (float*)dhead, partial);
  else ppo_loss_kernel<bf16, float><<<grid, LP_ROWS, smem, st>>>(m, A, head, idx, act, adv, ret, logp_old, eps, c1, c2, norm_adv, red, (bf16*)dhead, partial); }
  ProfScope ps2(K_STATS, st, 1, 0.0, (double)grid * 40);
  stats_final_kernel<<<1, 256, 0, st>>>(m, grid, partial, 1, c1, c2, 0, stats);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

// ------------------------------------------------------------------------------------------------
// O9 (A12, A13): ||g||_2 by a two-stage fixed-order fp64 reduction over fixed 4096-element chunks,
// then g c / max(||g||, c) and Adam, 16-byte vector loads and stores.
// ------------------------------------------------------------------------------------------------
constexpr int NORM_CHUNK = 4096;

__global__ void __launch_bounds__(256) sqnorm_partial_kernel(size_t P, const float* __restrict__ g, double* __restrict__ partial) {
  __shared__ double sh[256];
  size_t base = (size_t)blockIdx.x * NORM_CHUNK;
  double v = 0.0;
#pragma unroll
  for (int i = 0; i < NORM_CHUNK / 1024; ++i) {
    size_t e = base + ((size_t)i * 256 + threadIdx.x) * 4;
    if (e + 3 < P) { float4 x = *reinterpret_cast<const float4*>(g + e); v += (double)x.x * x.x + (double)x.y * x.y + (double)x.z * x.z + (double)x.w * x.w; }
    else for (size_t j = e; j < P; ++j) v += (double)g[j] * g[j];
  }
  double s = block_sum<256>(v, sh);
  if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

// gn1 = slot 4 of the update's stats record (or NULL).  errflag set (a tcgen05 pipeline timed out somewhere in this step): the
// norm becomes NaN, which makes the optimizer kernel skip the update, the record's loss and grad norm read NaN, and the host
// word is raised (cleanba.h, asynchronous errors).
__global__ void __launch_bounds__(256) sqnorm_final_kernel(int nparts, const double* __restrict__ partial, double* __restrict__ norm_out, float* __restrict__ gn0, float* __restrict__ gn1,
                                                           const int* __restrict__ errflag, int* errhost) {
  __shared__ double sh[256];
  double v = 0.0;
  for (int i = threadIdx.x; i < nparts; i += 256) v += partial[i];
  double s = block_sum<256>(v, sh);
  if (threadIdx.x == 0) {
    double n = sqrt(s);
    if (errflag && *errflag) { n = (double)NAN; if (gn1) gn1[-4] = NAN; if (errhost) *errhost = *errflag; }
    *norm_out = n; if (gn0) *gn0 = (float)n; if (gn1) *gn1 = (float)n;
  }
}

__device__ __forceinline__ void adam_one(float& th, float& m, float& v, float g, float scale, float b1, float omb1, float b2, float omb2,
                                         float ibc1, float ibc2, float lr, float eps) {
  g *= scale;
  m = fmaf(b1, m, omb1 * g);
  v = fmaf(b2, v, omb2 * g * g);
  th -= lr * (m * ibc1) / (sqrtf(v * ibc2) + eps);
}

__global__ void __launch_bounds__(256) adam_kernel(size_t P, float* __restrict__ th, float* __restrict__ m, float* __restrict__ v, const float* __restrict__ g,
                                                   const double* __restrict__ norm, float max_norm, float b1, float omb1, float b2, float omb2, float ibc1,
                                                   float ibc2, float lr, float eps) {
  double n = *norm;
  if (n != n) return;      // poisoned step: leave params and optimizer state untouched
  float scale = (float)((double)max_norm / fmax(n, (double)max_norm));
  size_t nv = P / 4;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < nv; i += (size_t)gridDim.x * blockDim.x) {
    float4 t4 = reinterpret_cast<float4*>(th)[i], m4 = reinterpret_cast<float4*>(m)[i], v4 = reinterpret_cast<float4*>(v)[i];
    float4 g4 = reinterpret_cast<const float4*>(g)[i];
    adam_one(t4.x, m4.x, v4.x, g4.x, scale, b1, omb1, b2, omb2, ibc1, ibc2, lr, eps);
    adam_one(t4.y, m4.y, v4.y, g4.y, scale, b1, omb1, b2, omb2, ibc1, ibc2, lr, eps);
    adam_one(t4.z, m4.z, v4.z, g4.z, scale, b1, omb1, b2, omb2, ibc1, ibc2, lr, eps);
    adam_one(t4.w, m4.w, v4.w, g4.w, scale, b1, omb1, b2, omb2, ibc1, ibc2, lr, eps);
    reinterpret_cast<float4*>(th)[i] = t4; reinterpret_cast<float4*>(m)[i] = m4; reinterpret_cast<float4*>(v)[i] = v4;
  }
  if (blockIdx.x == 0 && threadIdx.x < (P & 3)) {
    size_t i = nv * 4 + threadIdx.x;
    adam_one(th[i], m[i], v[i], g[i], scale, b1, omb1, b2, omb2, ibc1, ibc2, lr, eps);
  }
}

// A22: RMSprop with eps inside the root; nu_0 = 0.  16-byte loads and stores like adam_kernel.
__device__ __forceinline__ void rms_one(float& th, float& nu, float g, float scale, float decay, float omd, float lr, float eps) {
  const float gi = g * scale;
  nu = fmaf(decay, nu, omd * gi * gi);
  th -= lr * gi / sqrtf(nu + eps);
}
__global__ void __launch_bounds__(256) rmsprop_kernel(size_t P, float* __restrict__ th, float* __restrict__ nu, const float* __restrict__ g,
                                                      const double* __restrict__ norm, float max_norm, float decay, float omd, float lr, float eps) {
  const double n = *norm;
  if (n != n) return;      // poisoned step
  const float scale = (float)((double)max_norm / fmax(n, (double)max_norm));
  const size_t nv = P / 4;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < nv; i += (size_t)gridDim.x * blockDim.x) {
    float4 t4 = reinterpret_cast<float4*>(th)[i], n4 = reinterpret_cast<float4*>(nu)[i];
    const float4 g4 = reinterpret_cast<const float4*>(g)[i];
    rms_one(t4.x, n4.x, g4.x, scale, decay, omd, lr, eps); rms_one(t4.y, n4.y, g4.y, scale, decay, omd, lr, eps);
    rms_one(t4.z, n4.z, g4.z, scale, decay, omd, lr, eps); rms_one(t4.w, n4.w, g4.w, scale, decay, omd, lr, eps);
    reinterpret_cast<float4*>(th)[i] = t4; reinterpret_cast<float4*>(nu)[i] = n4;
  }
  if (blockIdx.x == 0 && threadIdx.x < (P & 3)) {
    const size_t i = nv * 4 + threadIdx.x;
    rms_one(th[i], nu[i], g[i], scale, decay, omd, lr, eps);
  }
}

int launch_clip_rmsprop(size_t P, float* params, float* nu, const float* g, float lr, float decay, float eps, float max_norm, float* grad_norm,
                        float* stats_slot, void* scratch, cudaStream_t st, const int* errflag, int* errhost) {
  if (P == 0) return CB_OK;
  int nparts = (int)((P + NORM_CHUNK - 1) / NORM_CHUNK);
  double* partial = (double*)scratch + 1; double* norm = (double*)scratch;
  { ProfScope ps(K_SQNORM, st, 2, 0.0, (double)P * 4);
  sqnorm_partial_kernel<<<nparts, 256, 0, st>>>(P, g, partial);
  sqnorm_final_kernel<<<1, 256, 0, st>>>(nparts, partial, norm, grad_norm, stats_slot, errflag, errhost); }
  ProfScope ps(K_ADAM, st, 1, 0.0, (double)P * 20);
  int grid = (int)std::min<size_t>((P / 4 + 255) / 256, (size_t)148 * 8); if (grid < 1) grid = 1;
  rmsprop_kernel<<<grid, 256, 0, st>>>(P, params, nu, g, norm, max_norm, decay, (float)(1.0 - (double)decay), lr, eps);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

// env group [b0, b0+Bm) of a [T,B] rollout: frame indices of its (T+1) x Bm observations (t-major) and contiguous copies
// of its per-step data (A21)
__global__ void gather_traj_kernel(int T, int B, int b0, int Bm, const int32_t* __restrict__ act, const float* __restrict__ rew,
                                   const uint8_t* __restrict__ dones, const float* __restrict__ logmu, int32_t* __restrict__ fidx,
                                   int32_t* __restrict__ act_m, float* __restrict__ rew_m, uint8_t* __restrict__ dones_m, float* __restrict__ logmu_m) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (T + 1) * Bm) return;
  const int t = i / Bm, b = i - t * Bm, src = t * B + b0 + b;
  fidx[i] = src;
  if (t < T) { act_m[i] = act[src]; rew_m[i] = rew[src]; dones_m[i] = dones[src]; logmu_m[i] = logmu[src]; }
}
int launch_gather_traj(int T, int B, int b0, int Bm, const int32_t* act, const float* rew, const uint8_t* dones, const float* logmu, int32_t* fidx,
                       int32_t* act_m, float* rew_m, uint8_t* dones_m, float* logmu_m, cudaStream_t st) {
  ProfScope ps(K_HEAD_MISC, st);
  gather_traj_kernel<<<((T + 1) * Bm + 127) / 128, 128, 0, st>>>(T, B, b0, Bm, act, rew, dones, logmu, fidx, act_m, rew_m, dones_m, logmu_m);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

size_t clip_adam_scratch_bytes(size_t P) { return (((P + NORM_CHUNK - 1) / NORM_CHUNK) + 2) * sizeof(double); }

int launch_clip_adam(size_t P, float* params, float* m, float* v, const float* g, uint64_t k, float lr, float b1, float b2, float eps,
                     float max_norm, float* grad_norm, float* stats_slot, void* scratch, cudaStream_t st, const int* errflag, int* errhost) {
  if (P == 0) return CB_OK;
  int nparts = (int)((P + NORM_CHUNK - 1) / NORM_CHUNK);
  double* partial = (double*)scratch + 1; double* norm = (double*)scratch;
  { ProfScope ps(K_SQNORM, st, 2, 0.0, (double)P * 4);
  sqnorm_partial_kernel<<<nparts, 256, 0, st>>>(P, g, partial);
  sqnorm_final_kernel<<<1, 256, 0, st>>>(nparts, partial, norm, grad_norm, stats_slot, errflag, errhost); }
  double bc1 = 1.0 - pow((double)b1, (double)k), bc2 = 1.0 - pow((double)b2, (double)k);
  int grid = (int)std::min<size_t>((P / 4 + 255) / 256, (size_t)148 * 8); if (grid < 1) grid = 1;
  ProfScope ps(K_ADAM, st, 1, 0.0, (double)P * 28);
  adam_kernel<<<grid, 256, 0, st>>>(P, params, m, v, g, norm, max_norm, b1, (float)(1.0 - (double)b1), b2, (float)(1.0 - (double)b2),
                                    (float)(1.0 / bc1), (float)(1.0 / bc2), lr, eps);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

}  // namespace cb
