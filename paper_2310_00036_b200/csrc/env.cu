// Seeded synthetic environment on the device: the stand-in for `E.step(a_t) -> s_next, r_t, d_next` (Alg. 1 l.9; EnvPool
// Atari in the paper) that lets a rollout of the actor/learner pipeline (pipeline.cu) stay on the GPU.  Input
// generation, not method arithmetic: the definition is paper_2310_00036_b200/synth.py `BlobEnv` (integer arithmetic only), restated
// here and tested bit for bit against it (tests/test_gpu_pipeline.py).
#include "common.cuh"

namespace cb {

constexpr int ENV_NB = 4;
constexpr int ENV_NS = 6 * ENV_NB + 1;      // per blob: cx, cy, vx, vy, amp, R; then the episode counter

__host__ __device__ __forceinline__ uint32_t mix32(uint32_t x) { x ^= x >> 16; x *= 0x7FEB352Du; x ^= x >> 15; x *= 0x846CA68Bu; x ^= x >> 16; return x; }
__device__ __forceinline__ uint32_t env_hash(uint32_t s, uint32_t a, uint32_t b, uint32_t c) { return mix32(s ^ mix32(a ^ mix32(b ^ mix32(c)))); }

__device__ __forceinline__ void env_spawn(int* st, uint32_t s, uint32_t e, uint32_t key, int H, int W) {
  for (int k = 0; k < ENV_NB; ++k) {
    st[6 * k + 0] = (int)(env_hash(s, e, key, 8 * k + 0) % (uint32_t)W); st[6 * k + 1] = (int)(env_hash(s, e, key, 8 * k + 1) % (uint32_t)H);
    st[6 * k + 2] = (int)(env_hash(s, e, key, 8 * k + 2) % 5u) - 2;         st[6 * k + 3] = (int)(env_hash(s, e, key, 8 * k + 3) % 5u) - 2;
    st[6 * k + 4] = 40 + (int)(env_hash(s, e, key, 8 * k + 4) % 161u);      st[6 * k + 5] = 6 + (int)(env_hash(s, e, key, 8 * k + 5) % 15u);
  }
}
__device__ __forceinline__ uint8_t env_pixel(const int* st, uint32_t s, uint32_t e, uint32_t g, int y, int x, int W) {
  int v = 0;
#pragma unroll
  for (int k = 0; k < ENV_NB; ++k) {
    const int R = st[6 * k + 5];
    v += st[6 * k + 4] * max(0, R - abs(x - st[6 * k])) * max(0, R - abs(y - st[6 * k + 1])) / (R * R);
  }
  v += (int)(env_hash(s, e, g, 1000u + (uint32_t)(y * W + x)) & 15u);
  return (uint8_t)min(v, 255);
}

// one block per env.  obs_in: the env's current stack [C,H,W] (unused by a reset); out0 / out1 (nullable): where the next stack goes.
template <bool RESET>
__global__ void __launch_bounds__(256) env_kernel(uint32_t s, int C, int H, int W, uint32_t g, const int32_t* __restrict__ actions, int32_t* __restrict__ state,
                                                  const uint8_t* __restrict__ obs_in, uint8_t* __restrict__ out0, uint8_t* __restrict__ out1,
                                                  float* __restrict__ rewards, uint8_t* __restrict__ dones) {
  __shared__ int st[ENV_NS]; __shared__ int s_done;
  const uint32_t e = blockIdx.x;
  if (threadIdx.x == 0) {
    if (RESET) {
      st[ENV_NS - 1] = 0; env_spawn(st, s, e, 0xFFFFFFFFu, H, W); s_done = 1;
    } else {
      for (int i = 0; i < ENV_NS; ++i) st[i] = state[(size_t)e * ENV_NS + i];
      const int a = actions[e], speed = a < 9 ? 2 : 1;
      st[0] = min(max(st[0] + (a % 3 - 1) * speed, 0), W - 1); st[1] = min(max(st[1] + ((a / 3) % 3 - 1) * speed, 0), H - 1);
      for (int k = 1; k < ENV_NB; ++k)
        for (int ax = 0; ax < 2; ++ax) {
          const int lim = ax ? H : W, p = st[6 * k + ax] + st[6 * k + 2 + ax];
          if (p < 0 || p >= lim) st[6 * k + 2 + ax] = -st[6 * k + 2 + ax];
          st[6 * k + ax] = min(max(p, 0), lim - 1);
        }
      const bool catch_ = abs(st[0] - st[6]) + abs(st[1] - st[7]) <= 8, hit = abs(st[0] - st[12]) + abs(st[1] - st[13]) <= 5;
      if (catch_) { st[6] = (int)(env_hash(s, e, g, 100u) % (uint32_t)W); st[7] = (int)(env_hash(s, e, g, 101u) % (uint32_t)H); }
      const bool done = hit || (env_hash(s, e, g, 102u) % 64u == 0u);
      rewards[e] = hit ? -1.f : (catch_ ? 1.f : 0.f); dones[e] = done ? 1 : 0;
      if (done) { st[ENV_NS - 1] += 1; env_spawn(st, s, e, g * 2654435761u + (uint32_t)st[ENV_NS - 1], H, W); }
      s_done = done ? 1 : 0;
    }
    for (int i = 0; i < ENV_NS; ++i) state[(size_t)e * ENV_NS + i] = st[i];
  }
  __syncthreads();
  const size_t fs = (size_t)C * H * W, plane = (size_t)H * W;
  const bool all = s_done != 0;
  for (int p = threadIdx.x; p < H * W; p += blockDim.x) {
    const uint8_t px = env_pixel(st, s, e, RESET ? 0xFFFFFFFFu : g, p / W, p % W, W);
    for (int c = 0; c < C; ++c) {
      const uint8_t v = (all || c == C - 1) ? px : obs_in[e * fs + (size_t)(c + 1) * plane + p];
      if (out0) out0[e * fs + (size_t)c * plane + p] = v;
      if (out1) out1[e * fs + (size_t)c * plane + p] = v;
    }
  }
}

static inline uint32_t seed32(uint64_t seed) { return mix32((uint32_t)seed) ^ (uint32_t)(seed >> 32); }

int launch_env_reset(uint64_t seed, int B, int C, int H, int W, int32_t* state, uint8_t* obs, cudaStream_t st) {
  if (B <= 0) return CB_OK;
  ProfScope ps(K_ENV, st);
  env_kernel<true><<<B, 256, 0, st>>>(seed32(seed), C, H, W, 0u, nullptr, state, nullptr, obs, nullptr, nullptr, nullptr);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}
int launch_env_step(uint64_t seed, int B, int C, int H, int W, uint32_t g, const int32_t* actions, int32_t* state, const uint8_t* obs_in, uint8_t* out0,
                    uint8_t* out1, float* rewards, uint8_t* dones, cudaStream_t st) {
  if (B <= 0) return CB_OK;
  ProfScope ps(K_ENV, st);
  env_kernel<false><<<B, 256, 0, st>>>(seed32(seed), C, H, W, g, actions, state, obs_in, out0, out1, rewards, dones);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

}  // namespace cb

using namespace cb;

extern "C" {

size_t cb_env_state_ints(void) { return ENV_NS; }

int cb_env_reset(uint64_t seed, int B, int C, int H, int W, int32_t* state, uint8_t* obs, void* stream) {
  if (B < 0 || C < 1 || H < 1 || W < 1 || !state || !obs) { set_error("bad argument"); return CB_EINVAL; }
  return launch_env_reset(seed, B, C, H, W, state, obs, (cudaStream_t)stream);
}
int cb_env_step(uint64_t seed, int B, int C, int H, int W, uint32_t global_step, const int32_t* actions, int32_t* state, const uint8_t* obs_in,
                uint8_t* obs_out, float* rewards, uint8_t* dones, void* stream) {
  if (B < 0 || C < 1 || H < 1 || W < 1 || !state || !obs_in || !obs_out || !actions || !rewards || !dones || obs_in == obs_out) { set_error("bad argument"); return CB_EINVAL; }
  return launch_env_step(seed, B, C, H, W, global_step, actions, state, obs_in, obs_out, nullptr, rewards, dones, (cudaStream_t)stream);
}

}  // extern "C"
