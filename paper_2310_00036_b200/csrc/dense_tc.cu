// tcgen05 / TMEM GEMMs for the dense trunk (fc layer) in CB_PREC_BF16_TC:
//   MODE 0  forward:  hid[f][n]  = sum_k relu(A[f][k]) * Wf[k][n] + b[n]        (M = frames,   contraction = features)
//   MODE 1  wgrad:    dW[k][n]   = sum_f relu(A[f][k]) * dY[f][n]               (M = features, contraction = frames)
//   MODE 2  dgrad:    dA[f][k]   = [A[f][k] > 0] sum_n dY[f][n] * Wf[k][n]      (M = frames,   contraction = outputs)
// A is the NHWC-flattened feature map [F][K] (bf16), Wf the forward weight pack [K][N], dY [F][N].
// Operands are staged by 8 loader warps as 16-byte units into padded planes so that they are canonical
// no-swizzle UMMA layouts (rows of a core matrix 16 B apart): forward A is K-major (LBO = plane), every other
// operand is MN-major (LBO = 128 B, SBO = plane).  4-stage mbarrier pipeline: loaders run ahead of the
// single MMA-issuing thread; the fp32 accumulator [128 x BN] lives in TMEM; warps 0-3 drain it.
#include "common.cuh"
#include "tc_ptx.cuh"

namespace cb {
namespace dn {
using namespace ptx;

struct Args {
  const bf16* A;      // MODE 0/1: features [F][K];  MODE 2: dY [F][N]
  const bf16* B;      // MODE 0/2: Wf [K][N];  MODE 1: dY [F][N]
  const bf16* mask;   // MODE 2: feature pre-activations [F][K] gating the result (nullable)
  const float* bias;  // MODE 0
  bf16* out;          // MODE 0: [F][N]
  float* grad;        // MODE 1: canonical fp32 gradient buffer
  int F, K, N, relu_in;
  float* part; int ksplit;      // MODE 0 with ksplit > 1: fp32 partial sums [ksplit][F][N] instead of out
  int H, W, C; size_t w_off;   // MODE 1: feature k = (y*W + x)*C + c  ->  canonical fc.w index n*K + (c*H + y)*W + x
  int* error_flag;
};

constexpr int NLOAD = 256, BK = 64, NSTAGE = 4;
constexpr uint32_t PB = BK * 16 + 16;

__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}\n" :: "r"(bar) : "memory");
}
__device__ __forceinline__ uint4 relu8(uint4 v) {
  __nv_bfloat162* h = reinterpret_cast<__nv_bfloat162*>(&v);
  const __nv_bfloat162 z = __float2bfloat162_rn(0.f);
#pragma unroll
  for (int k = 0; k < 4; ++k) h[k] = __hmax2(h[k], z);
  return v;
}

template <int MODE, int BN>
__global__ void __launch_bounds__(NLOAD + 32) dense_tc_kernel(const Args a) {
  extern __shared__ __align__(128) uint8_t smem[];
  constexpr uint32_t PA = (MODE != 1 ? 128 : BK) * 16 + 16;
  constexpr int APL = MODE != 1 ? BK / 8 : 16, BPL = MODE == 2 ? BK / 8 : BN / 8;
  constexpr uint32_t PBK = BN * 16 + 16;                 // MODE 2: K-major B planes [contraction/8][BN rows][16 B]
  constexpr uint32_t STAGE = APL * PA + BPL * (MODE == 2 ? PBK : PB);
  constexpr uint32_t TCOLS = BN < 32 ? 32 : BN;
  __shared__ __align__(8) uint64_t bars[2 * NSTAGE + 1];
  __shared__ uint32_t tmem_base_smem;
  const int tid = threadIdx.x, warp = tid >> 5;
  const uint32_t bar0 = smem_u32(&bars[0]);
  if (tid == 0) {
    for (int i = 0; i < 2 * NSTAGE + 1; ++i) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" :: "r"(bar0 + 8u * i) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  if (warp == NLOAD / 32) tmem_alloc(smem_u32(&tmem_base_smem), TCOLS);
  tc_fence_before(); __syncthreads(); tc_fence_after();
  const uint32_t tmem_base = tmem_base_smem;
  const int m0 = blockIdx.x * 128, n0 = blockIdx.y * BN;
  const int L = MODE == 0 ? a.K : (MODE == 1 ? a.F : a.N);      // contraction length
  const int lda = MODE == 2 ? a.N : a.K;                         // row length of A
  const int all_tiles = (L + BK - 1) / BK;
  const int per_z = (all_tiles + (int)gridDim.z - 1) / (int)gridDim.z;
  const int tbeg = (int)blockIdx.z * per_z, ntiles = max(0, min(all_tiles, tbeg + per_z) - tbeg);      // this CTA's k-tiles

  if (warp < NLOAD / 32) {
    for (int t = 0; t < ntiles; ++t) {
      const int s = t % NSTAGE, use = t / NSTAGE, l0 = (tbeg + t) * BK;
      if (use > 0 && !mbar_wait(bar0 + 8u * (NSTAGE + s), (uint32_t)((use - 1) & 1))) { if (a.error_flag) *a.error_flag = 5; }
      uint8_t* as = smem + (size_t)s * STAGE; uint8_t* bs = as + APL * PA;
      // ---- A tile ----
      constexpr int AWORK = 128 * (BK / 8);               // 16-byte units (both modes: 128 x 64 elements)
#pragma unroll
      for (int i0 = 0; i0 < AWORK; i0 += NLOAD) {
        const int i = i0 + tid;
        uint4 v = make_uint4(0, 0, 0, 0); uint32_t dst;
        if (MODE != 1) {
          const int row = i >> 3, j = i & 7, f = m0 + row, k = l0 + 8 * j;
          dst = (uint32_t)j * PA + (uint32_t)row * 16u;
          if (f < a.F && k < L) v = *reinterpret_cast<const uint4*>(a.A + (size_t)f * lda + k);
        } else {
          const int frow = i >> 4, g = i & 15, f = l0 + frow, k = m0 + 8 * g;
          dst = (uint32_t)g * PA + (uint32_t)frow * 16u;
          if (f < a.F && k < a.K) v = *reinterpret_cast<const uint4*>(a.A + (size_t)f * a.K + k);
        }
        if (MODE != 2 && a.relu_in) v = relu8(v);
        *reinterpret_cast<uint4*>(as + dst) = v;
      }
      if (MODE == 2) {
        // ---- B tile (K-major): rows = outputs k = n0 .. n0+BN of Wf [K][N], contraction columns l0 .. l0+BK ----
        for (int i = tid; i < BN * (BK / 8); i += NLOAD) {
          const int row = i >> 3, j = i & 7, k = n0 + row, n = l0 + 8 * j;
          uint4 v = make_uint4(0, 0, 0, 0);
          if (k < a.K && n < a.N) v = *reinterpret_cast<const uint4*>(a.B + (size_t)k * a.N + n);
          *reinterpret_cast<uint4*>(bs + (uint32_t)j * PBK + (uint32_t)row * 16u) = v;
        }
      }
      // ---- B tile: BK rows of [rows][N] starting at row l0, columns n0 .. n0+BN ----
      constexpr int BWORK = MODE == 2 ? 0 : BK * BPL;
      for (int i = tid; i < BWORK; i += NLOAD) {
        const int r = i / BPL, g = i - r * BPL, row = l0 + r, n = n0 + 8 * g;
        uint4 v = make_uint4(0, 0, 0, 0);
        if (row < L && n < a.N) v = *reinterpret_cast<const uint4*>(a.B + (size_t)row * a.N + n);
        *reinterpret_cast<uint4*>(bs + (uint32_t)g * PB + (uint32_t)r * 16u) = v;
      }
      fence_async_smem();
      asm volatile("bar.sync 1, %0;\n" :: "n"(NLOAD) : "memory");
      if (tid == 0) mbar_arrive(bar0 + 8u * s);
    }
    if (warp < 4) {
      if (ntiles > 0 && !mbar_wait(bar0 + 8u * (2 * NSTAGE), 0u)) { if (a.error_flag) *a.error_flag = 5; }
      tc_fence_after();
      const int row = m0 + tid;
#pragma unroll
      for (int c0 = 0; c0 < BN; c0 += 16) {
        float v[16];
        tmem_ld16(tmem_base + ((uint32_t)(warp * 32) << 16) + (uint32_t)c0, v);
        const int n = n0 + c0;
        if (n >= (MODE == 2 ? a.K : a.N)) continue;
        if (MODE == 2) {
          if (row >= a.F) continue;
          const size_t o = (size_t)row * a.K + n;
          if (a.mask) {
            uint4 s0 = *reinterpret_cast<const uint4*>(a.mask + o), s1 = *reinterpret_cast<const uint4*>(a.mask + o + 8);
            const bf16* h0 = reinterpret_cast<const bf16*>(&s0); const bf16* h1 = reinterpret_cast<const bf16*>(&s1);
#pragma unroll
            for (int i = 0; i < 8; ++i) { if (!(__bfloat162float(h0[i]) > 0.f)) v[i] = 0.f; if (!(__bfloat162float(h1[i]) > 0.f)) v[8 + i] = 0.f; }
          }
          uint4 o0, o1;
          __nv_bfloat162* p0 = reinterpret_cast<__nv_bfloat162*>(&o0); __nv_bfloat162* p1 = reinterpret_cast<__nv_bfloat162*>(&o1);
#pragma unroll
          for (int i = 0; i < 4; ++i) { p0[i] = __floats2bfloat162_rn(v[2 * i], v[2 * i + 1]); p1[i] = __floats2bfloat162_rn(v[8 + 2 * i], v[8 + 2 * i + 1]); }
          *reinterpret_cast<uint4*>(a.out + o) = o0;
          *reinterpret_cast<uint4*>(a.out + o + 8) = o1;
        } else if (MODE == 0) {
          if (row >= a.F) continue;
          if (a.ksplit > 1) {
#pragma unroll
            for (int i = 0; i < 16; ++i) a.part[((size_t)blockIdx.z * a.F + row) * a.N + n + i] = ntiles > 0 ? v[i] : 0.f;
            continue;
          }
#pragma unroll
          for (int i = 0; i < 16; ++i) v[i] += a.bias[n + i];
          uint4 o0, o1;
          __nv_bfloat162* p0 = reinterpret_cast<__nv_bfloat162*>(&o0); __nv_bfloat162* p1 = reinterpret_cast<__nv_bfloat162*>(&o1);
#pragma unroll
          for (int i = 0; i < 4; ++i) { p0[i] = __floats2bfloat162_rn(v[2 * i], v[2 * i + 1]); p1[i] = __floats2bfloat162_rn(v[8 + 2 * i], v[8 + 2 * i + 1]); }
          *reinterpret_cast<uint4*>(a.out + (size_t)row * a.N + n) = o0;
          *reinterpret_cast<uint4*>(a.out + (size_t)row * a.N + n + 8) = o1;
        } else {
          if (row >= a.K) continue;
          const int c = row % a.C, pix = row / a.C, y = pix / a.W, x = pix - y * a.W;
          const size_t kc = ((size_t)c * a.H + y) * a.W + x;
#pragma unroll
          for (int i = 0; i < 16; ++i) a.grad[a.w_off + (size_t)(n + i) * a.K + kc] = v[i];
        }
      }
    }
  } else {      // warp NLOAD / 32: the whole warp runs the loop, one elected lane issues
    const uint32_t idesc = make_idesc(128, BN, MODE == 1 ? 1 : 0, MODE == 2 ? 0 : 1);
    for (int t = 0; t < ntiles; ++t) {
      const int s = t % NSTAGE, use = t / NSTAGE;
      if (!mbar_wait(bar0 + 8u * s, (uint32_t)(use & 1))) { if (a.error_flag) *a.error_flag = 5; }
      tc_fence_after();
      const uint32_t ab = smem_u32(smem + (size_t)s * STAGE), bb = ab + APL * PA;
#pragma unroll
      for (int ks = 0; ks < BK / 16; ++ks) {
        const uint64_t ad = MODE != 1 ? make_desc(ab + (uint32_t)(2 * ks) * PA, PA, 128u) : make_desc(ab + (uint32_t)ks * 256u, 128u, PA);
        const uint64_t bd = MODE == 2 ? make_desc(bb + (uint32_t)(2 * ks) * PBK, PBK, 128u) : make_desc(bb + (uint32_t)ks * 256u, 128u, PB);
        if (elect_one()) mma_f16(tmem_base, ad, bd, idesc, (t | ks) ? 1u : 0u);
      }
      if (elect_one()) mma_commit(bar0 + 8u * (NSTAGE + s));
      __syncwarp();
    }
    if (ntiles > 0 && elect_one()) mma_commit(bar0 + 8u * (2 * NSTAGE));
    __syncwarp();
  }
  tc_fence_before(); __syncthreads();
  if (warp == NLOAD / 32) tmem_dealloc(tmem_base, TCOLS);
}

// out[f][n] = bf16(sum_z part[z][f][n] + bias[n]), z in order
__global__ void dense_reduce_kernel(const float* __restrict__ part, int S, int F, int N, const float* __restrict__ bias, bf16* __restrict__ out) {
  size_t total = (size_t)F * N;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    float s = 0.f;
    for (int z = 0; z < S; ++z) s += part[(size_t)z * total + i];
    out[i] = __float2bfloat16_rn(s + bias[i % N]);
  }
}

// db[n] = sum_f dY[f][n]: 16 lanes per column, lane k sums frames [k*q, (k+1)*q) in order, then the 16 sums are added in
// lane order (fixed association => reproducible)
__global__ void colsum_kernel(const bf16* __restrict__ dy, int F, int N, float* __restrict__ out) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x, n = t >> 4, part = t & 15;
  const int q = (F + 15) / 16, f0 = part * q, f1 = min(F, f0 + q);
  float s = 0.f;
  if (n < N) {
#pragma unroll 8
    for (int f = f0; f < f1; ++f) s += __bfloat162float(dy[(size_t)f * N + n]);
  }
  float tot = s;
#pragma unroll
  for (int k = 1; k < 16; ++k) tot += __shfl_down_sync(0xffffffffu, s, k);
  if (part == 0 && n < N) out[n] = tot;
}

}  // namespace dn

bool dense_tc_supported(const Geom& g) {
  return g.Ho == 1 && g.Wo == 1 && g.kh == g.H && g.kw == g.W && g.p == 0 && g.Cin % 8 == 0 && g.Cout % 64 == 0;
}

template <int MODE, int BN>
static int launch_d(const dn::Args& a, dim3 grid, cudaStream_t st) {
  if (a.ksplit > 1) grid.z = a.ksplit;
  constexpr size_t PA = (MODE != 1 ? 128 : dn::BK) * 16 + 16;
  constexpr size_t smem = dn::NSTAGE * ((MODE != 1 ? dn::BK / 8 : 16) * PA + (MODE == 2 ? (dn::BK / 8) * (BN * 16 + 16) : (BN / 8) * dn::PB));
  { int rc = ensure_dyn_smem((const void*)dn::dense_tc_kernel<MODE, BN>, smem); if (rc) return rc; }
  dn::dense_tc_kernel<MODE, BN><<<grid, dn::NLOAD + 32, smem, st>>>(a);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

int launch_dense_fwd_tc(const Geom& g, int F, const bf16* A, const bf16* wf, const float* bias, bf16* out, bool relu_in, float* partial, int* error_flag, cudaStream_t st) {
  if (F <= 0) return CB_OK;
  const int K = g.H * g.W * g.Cin, N = g.Cout;
  const int ksplit = (F <= 1024 && partial) ? 8 : 1;      // few frames (actor side): split the contraction so that the grid fills the GPU
  dn::Args a{A, wf, nullptr, bias, out, nullptr, F, K, N, relu_in ? 1 : 0, partial, ksplit, g.H, g.W, g.Cin, 0, error_flag};
  int rc = launch_d<0, 32>(a, dim3((F + 127) / 128, (N + 31) / 32), st);
  if (rc || ksplit == 1) return rc;
  dn::dense_reduce_kernel<<<std::min((F * N + 255) / 256, 1184), 256, 0, st>>>(partial, ksplit, F, N, bias, out);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

int launch_dense_wgrad_tc(const Geom& g, const ParamMap& pm, int F, const bf16* A, const bf16* dy, bool relu_in, float* grad, int* error_flag, cudaStream_t st) {
  if (F <= 0) return CB_OK;
  const int K = g.H * g.W * g.Cin, N = g.Cout;
  dn::Args a{A, dy, nullptr, nullptr, nullptr, grad, F, K, N, relu_in ? 1 : 0, nullptr, 1, g.H, g.W, g.Cin, pm.w_off, error_flag};
  int rc = launch_d<1, 64>(a, dim3((K + 127) / 128, (N + 63) / 64), st);
  if (rc) return rc;
  dn::colsum_kernel<<<(16 * N + 255) / 256, 256, 0, st>>>(dy, F, N, grad + pm.b_off);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

// dgrad of the fc layer: dx [F][K] = gate(dY [F][N] . Wf^T), gated by the stored feature pre-activations
int launch_dense_dgrad_tc(const Geom& g, int F, const bf16* dy, const bf16* wf, const bf16* mask, bf16* dx, int* error_flag, cudaStream_t st) {
  if (F <= 0) return CB_OK;
  const int K = g.H * g.W * g.Cin, N = g.Cout;
  dn::Args a{dy, wf, mask, nullptr, dx, nullptr, F, K, N, 0, nullptr, 1, g.H, g.W, g.Cin, 0, error_flag};
  return launch_d<2, 64>(a, dim3((F + 127) / 128, (K + 63) / 64), st);
}

}  // namespace cb
