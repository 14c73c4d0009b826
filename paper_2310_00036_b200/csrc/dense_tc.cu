// tcgen05 / TMEM GEMMs for the dense trunk (fc layer) in CB_PREC_BF16_TC, fed by TMA:
//   MODE 0  forward:  hid[f][n]  = sum_k A[f][k] * Wt[n][k] + b[n]               (M = frames,   N = outputs,  contraction = features)
//   MODE 2  dgrad:    dA[f][k]   = [A[f][k] > 0] sum_n dY[f][n] * Wf[k][n]       (M = frames,   N = features, contraction = outputs)
//   wgrad:            dW[k][n]   = sum_f A[f][k] * dY[f][n]                      (M = features, N = outputs,  contraction = frames)
// A is the NHWC-flattened feature map [F][K] (bf16; the producing layer stores it through its ReLU, api.cu), Wt / Wf the two weight
// packs ([N][K] and [K][N]), dY [F][N].  Every operand tile is landed by 2-D `cp.async.bulk.tensor` boxes of 64 columns (128 bytes) in
// the 128-byte swizzle pattern, i.e. directly in the canonical swizzled UMMA layout: K-major for MODE 0 / 2 (the contraction index is
// the contiguous one in memory), MN-major for the weight gradient (frames are the rows of both operands; LBO = one 64-column block).
// Out-of-range rows / columns of a box are zero-filled by the TMA unit, so ragged F and K need no special case.  A CTA owns a
// [128 x 256] accumulator in TMEM; warp 0 produces (4-stage mbarrier ring), warp 1 issues the MMAs, warps 2-5 drain the accumulator.
// MODE 0 splits the contraction over gridDim.z CTAs (a constant of the layer, never of F, so that a frame's result does not depend on
// the batch it is in) and a second kernel adds the partials in split order, the bias, and rounds to bf16.
#include "common.cuh"
#include "tc_ptx.cuh"
#include "tma.cuh"

namespace cb {
namespace dn {
using namespace ptx;

struct Args {
  const float* bias;  // MODE 0 (applied by the reduce kernel)
  const bf16* mask;   // MODE 2: feature map [F][K] whose sign gates the result (nullable)
  bf16* out;          // MODE 2: dA [F][K]
  float* part;        // MODE 0: fp32 partial sums [ksplit][F][N]
  float* grad;        // wgrad: canonical fp32 gradient buffer
  int F, K, N;
  int H, W, C; size_t w_off;   // wgrad: feature k = (y*W + x)*C + c  ->  canonical fc.w index n*K + (c*H + y)*W + x
  int* error_flag;
};

constexpr int BK = 64, NST = 4, BM = 128, BN = 256, NTHREADS = 6 * 32;
constexpr uint32_t A_BYTES = BM * BK * 2, B_BYTES = BN * BK * 2, STAGE = A_BYTES + B_BYTES, SMEM = NST * STAGE + 1024;
// MODE 2 contracts over the layer's outputs (4 tiles for fc = 256): two stages, so that two CTAs share an SM and overlap their load / MMA / drain phases
constexpr int NST2 = 2; constexpr uint32_t SMEM2 = NST2 * STAGE + 1024;
constexpr uint32_t BLK = 64 * 128;      // one box: 64 rows of 128 bytes

__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n"
               :: "r"(dst), "l"((uint64_t)map), "r"(c0), "r"(c1), "r"(bar) : "memory");
}
// SW128 descriptor: start address, LBO (bytes; MN-major: distance between 64-element blocks along M / N), SBO = 1024 B (8 rows of 128 B)
__device__ __forceinline__ uint64_t sw128_desc(uint32_t saddr, uint32_t lbo_bytes) {
  return (uint64_t)((saddr >> 4) & 0x3FFFu) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFFu) << 16) | ((uint64_t)(1024u >> 4) << 32) | ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}

// MODE 0 / 2: both operands K-major.  amap: rows = frames, columns = contraction; bmap: rows = N index, columns = contraction.
template <int MODE>
__global__ void __launch_bounds__(NTHREADS) dense_kmajor_kernel(const Args a, const __grid_constant__ CUtensorMap amap, const __grid_constant__ CUtensorMap bmap) {
  constexpr int NST = MODE == 2 ? NST2 : dn::NST;
  extern __shared__ __align__(128) uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t bars[2 * NST + 1];
  __shared__ uint32_t tmem_base_smem;
  const int tid = threadIdx.x, warp = tid >> 5;
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u, bar0 = smem_u32(&bars[0]);
  if (tid == 0) {
    for (int i = 0; i < 2 * NST + 1; ++i) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" :: "r"(bar0 + 8u * i) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    tma::prefetch_map(&amap); tma::prefetch_map(&bmap);
  }
  if (warp == 1) tmem_alloc(smem_u32(&tmem_base_smem), BN);
  tc_fence_before(); __syncthreads(); tc_fence_after();
  const uint32_t tmem_base = tmem_base_smem;
  const int m0 = blockIdx.x * BM, n0 = blockIdx.y * BN;
  const int L = MODE == 0 ? a.K : a.N;                                   // contraction length
  const int all_tiles = (L + BK - 1) / BK, per_z = (all_tiles + (int)gridDim.z - 1) / (int)gridDim.z;
  const int tbeg = (int)blockIdx.z * per_z, ntiles = max(0, min(all_tiles, tbeg + per_z) - tbeg);
  if (warp == 0) {
    // ================= TMA producer =================
    for (int t = 0; t < ntiles; ++t) {
      const int s = t % NST, use = t / NST, l0 = (tbeg + t) * BK;
      if (use > 0 && !mbar_wait(bar0 + 8u * (NST + s), (uint32_t)((use - 1) & 1))) { if (a.error_flag) *a.error_flag = 5; }
      if (elect_one()) {
        const uint32_t dst = sbase + (uint32_t)s * STAGE, full = bar0 + 8u * s;
        tma::arrive_expect_tx(full, STAGE);
        tma_load_2d(dst, &amap, l0, m0, full); tma_load_2d(dst + BLK, &amap, l0, m0 + 64, full);
#pragma unroll
        for (int j = 0; j < BN / 64; ++j) tma_load_2d(dst + A_BYTES + (uint32_t)j * BLK, &bmap, l0, n0 + 64 * j, full);
      }
      __syncwarp();
    }
  } else if (warp == 1) {
    // ================= MMA issuer =================
    const uint32_t idesc = make_idesc(BM, BN, 0, 0);
    for (int t = 0; t < ntiles; ++t) {
      const int s = t % NST, use = t / NST;
      if (!mbar_wait(bar0 + 8u * s, (uint32_t)(use & 1))) { if (a.error_flag) *a.error_flag = 5; }
      tc_fence_after();
      const uint32_t ab = sbase + (uint32_t)s * STAGE, bb = ab + A_BYTES;
#pragma unroll
      for (int ks = 0; ks < BK / 16; ++ks)      // 16 contraction elements = 32 bytes further along the swizzled 128-byte row
        if (elect_one()) mma_f16(tmem_base, sw128_desc(ab + 32u * ks, 16u), sw128_desc(bb + 32u * ks, 16u), idesc, (t | ks) ? 1u : 0u);
      if (elect_one()) mma_commit(bar0 + 8u * (NST + s));
      __syncwarp();
    }
    if (ntiles > 0 && elect_one()) mma_commit(bar0 + 8u * (2 * NST));
    __syncwarp();
  } else {
    // ================= epilogue: warp w drains TMEM lanes 32 (w % 4) .. +31 =================
    if (ntiles > 0 && !mbar_wait(bar0 + 8u * (2 * NST), 0u)) { if (a.error_flag) *a.error_flag = 5; }
    tc_fence_after();
    const int q = warp & 3, row = m0 + q * 32 + (tid & 31);
#pragma unroll 2
    for (int c0 = 0; c0 < BN; c0 += 16) {
      float v[16];
      tmem_ld16(tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)c0, v);
      const int n = n0 + c0;
      if (row >= a.F || n >= (MODE == 0 ? a.N : a.K)) continue;
      if (MODE == 0) {
        float4* dst = reinterpret_cast<float4*>(a.part + ((size_t)blockIdx.z * a.F + row) * a.N + n);
#pragma unroll
        for (int i = 0; i < 4; ++i) dst[i] = ntiles > 0 ? make_float4(v[4 * i], v[4 * i + 1], v[4 * i + 2], v[4 * i + 3]) : make_float4(0.f, 0.f, 0.f, 0.f);
      } else {
        const size_t o = (size_t)row * a.K + n;
        if (a.mask) {
          const uint4 s0 = *reinterpret_cast<const uint4*>(a.mask + o), s1 = *reinterpret_cast<const uint4*>(a.mask + o + 8);
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
      }
    }
  }
  tc_fence_before(); __syncthreads();
  if (warp == 1) tmem_dealloc(tmem_base, BN);
}

// Weight gradient: both operands MN-major.  amap = feature map [F][K], bmap = dY [F][N]; a stage holds 64 frames (contraction rows) of
// 128 feature columns (two boxes) and 256 output columns (four boxes).
__global__ void __launch_bounds__(NTHREADS) dense_wgrad_kernel(const Args a, const __grid_constant__ CUtensorMap amap, const __grid_constant__ CUtensorMap bmap) {
  extern __shared__ __align__(128) uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t bars[2 * NST + 1];
  __shared__ uint32_t tmem_base_smem;
  const int tid = threadIdx.x, warp = tid >> 5;
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u, bar0 = smem_u32(&bars[0]);
  if (tid == 0) {
    for (int i = 0; i < 2 * NST + 1; ++i) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" :: "r"(bar0 + 8u * i) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    tma::prefetch_map(&amap); tma::prefetch_map(&bmap);
  }
  if (warp == 1) tmem_alloc(smem_u32(&tmem_base_smem), BN);
  tc_fence_before(); __syncthreads(); tc_fence_after();
  const uint32_t tmem_base = tmem_base_smem;
  const int m0 = blockIdx.x * BM, n0 = blockIdx.y * BN;
  const int ntiles = (a.F + BK - 1) / BK;
  if (warp == 0) {
    for (int t = 0; t < ntiles; ++t) {
      const int s = t % NST, use = t / NST, f0 = t * BK;
      if (use > 0 && !mbar_wait(bar0 + 8u * (NST + s), (uint32_t)((use - 1) & 1))) { if (a.error_flag) *a.error_flag = 5; }
      if (elect_one()) {
        const uint32_t dst = sbase + (uint32_t)s * STAGE, full = bar0 + 8u * s;
        tma::arrive_expect_tx(full, STAGE);
        tma_load_2d(dst, &amap, m0, f0, full); tma_load_2d(dst + BLK, &amap, m0 + 64, f0, full);
#pragma unroll
        for (int j = 0; j < BN / 64; ++j) tma_load_2d(dst + A_BYTES + (uint32_t)j * BLK, &bmap, n0 + 64 * j, f0, full);
      }
      __syncwarp();
    }
  } else if (warp == 1) {
    const uint32_t idesc = make_idesc(BM, BN, 1, 1);
    for (int t = 0; t < ntiles; ++t) {
      const int s = t % NST, use = t / NST;
      if (!mbar_wait(bar0 + 8u * s, (uint32_t)(use & 1))) { if (a.error_flag) *a.error_flag = 5; }
      tc_fence_after();
      const uint32_t ab = sbase + (uint32_t)s * STAGE, bb = ab + A_BYTES;
#pragma unroll
      for (int ks = 0; ks < BK / 16; ++ks)      // 16 contraction rows = 16 * 128 bytes further down every block
        if (elect_one()) mma_f16(tmem_base, sw128_desc(ab + 2048u * ks, BLK), sw128_desc(bb + 2048u * ks, BLK), idesc, (t | ks) ? 1u : 0u);
      if (elect_one()) mma_commit(bar0 + 8u * (NST + s));
      __syncwarp();
    }
    if (ntiles > 0 && elect_one()) mma_commit(bar0 + 8u * (2 * NST));
    __syncwarp();
  } else {
    if (ntiles > 0 && !mbar_wait(bar0 + 8u * (2 * NST), 0u)) { if (a.error_flag) *a.error_flag = 5; }
    tc_fence_after();
    const int q = warp & 3, row = m0 + q * 32 + (tid & 31);      // feature index k
    const int c = row % a.C, pix = row / a.C, y = pix / a.W, x = pix - y * a.W;
    const size_t kc = ((size_t)c * a.H + y) * a.W + x;
#pragma unroll 2
    for (int c0 = 0; c0 < BN; c0 += 16) {
      float v[16];
      tmem_ld16(tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)c0, v);
      const int n = n0 + c0;
      if (row >= a.K || n >= a.N) continue;
#pragma unroll
      for (int i = 0; i < 16; ++i) a.grad[a.w_off + (size_t)(n + i) * a.K + kc] = ntiles > 0 ? v[i] : 0.f;
    }
  }
  tc_fence_before(); __syncthreads();
  if (warp == 1) tmem_dealloc(tmem_base, BN);
}

// out[f][n] = bf16(sum_z part[z][f][n] + bias[n]), z in order; four outputs per thread
__global__ void __launch_bounds__(256) dense_reduce_kernel(const float* __restrict__ part, int S, int F, int N, const float* __restrict__ bias, bf16* __restrict__ out) {
  const size_t total4 = (size_t)F * N / 4;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total4; i += (size_t)gridDim.x * blockDim.x) {
    float4 s = reinterpret_cast<const float4*>(part)[i];
    for (int z = 1; z < S; ++z) { const float4 p = reinterpret_cast<const float4*>(part)[(size_t)z * total4 + i]; s.x += p.x; s.y += p.y; s.z += p.z; s.w += p.w; }
    const float4 b = *reinterpret_cast<const float4*>(bias + (int)((i * 4) % (size_t)N));
    __nv_bfloat162 o[2] = {__floats2bfloat162_rn(s.x + b.x, s.y + b.y), __floats2bfloat162_rn(s.z + b.z, s.w + b.w)};
    *reinterpret_cast<uint2*>(out + i * 4) = *reinterpret_cast<const uint2*>(o);
  }
}

// db[n] = sum_f dY[f][n].  A block owns 8 columns (one 16-byte vector per frame): thread t sums frames t, t + 256, ... in order, then
// the 256 thread sums of a column are added by a fixed shared-memory tree (fixed association => reproducible).
__global__ void __launch_bounds__(256) colsum_kernel(const bf16* __restrict__ dy, int F, int N, float* __restrict__ out) {
  __shared__ float sh[256][9];
  const int n0 = blockIdx.x * 8;
  float s[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  for (int f = threadIdx.x; f < F; f += 256) {
    const uint4 v = *reinterpret_cast<const uint4*>(dy + (size_t)f * N + n0);
    const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&v);
#pragma unroll
    for (int k = 0; k < 4; ++k) { const float2 t = __bfloat1622float2(h[k]); s[2 * k] += t.x; s[2 * k + 1] += t.y; }
  }
#pragma unroll
  for (int k = 0; k < 8; ++k) sh[threadIdx.x][k] = s[k];
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if ((int)threadIdx.x < w) {
#pragma unroll
      for (int k = 0; k < 8; ++k) sh[threadIdx.x][k] += sh[threadIdx.x + w][k];
    }
    __syncthreads();
  }
  if (threadIdx.x < 8) out[n0 + threadIdx.x] = sh[0][threadIdx.x];
}

}  // namespace dn

bool dense_tc_supported(const Geom& g) {
  const int K = g.H * g.W * g.Cin;
  return g.Ho == 1 && g.Wo == 1 && g.kh == g.H && g.kw == g.W && g.p == 0 && g.Cin % 8 == 0 && K % 16 == 0 && g.Cout % 64 == 0 && tma::encode_fn() != nullptr;
}

// the contraction of the forward GEMM is split over this many CTAs whatever the batch size (A16: a frame's hidden vector must not
// depend on how many other frames are in the call)
constexpr int DENSE_KSPLIT = 8;
size_t dense_partial_elems(const Geom& g, long long frames) { return (size_t)DENSE_KSPLIT * (size_t)frames * g.Cout; }

static bool map2d(CUtensorMap* m, const void* base, int rows, int cols) { return tma::make_2d_map(m, base, rows, cols, 64, 64); }

int launch_dense_fwd_tc(const Geom& g, int F, const bf16* A, const bf16* wt, const float* bias, bf16* out, float* partial, int* error_flag, cudaStream_t st) {
  if (F <= 0) return CB_OK;
  const int K = g.H * g.W * g.Cin, N = g.Cout;
  CUtensorMap am, bm;
  if (!map2d(&am, A, F, K) || !map2d(&bm, wt, N, K)) { set_error("cuTensorMapEncodeTiled refused a dense-layer map"); return CB_ECUDA; }
  dn::Args a{bias, nullptr, nullptr, partial, nullptr, F, K, N, g.H, g.W, g.Cin, 0, error_flag};
  int rc = ensure_dyn_smem((const void*)dn::dense_kmajor_kernel<0>, dn::SMEM); if (rc) return rc;
  dn::dense_kmajor_kernel<0><<<dim3((F + dn::BM - 1) / dn::BM, (N + dn::BN - 1) / dn::BN, DENSE_KSPLIT), dn::NTHREADS, dn::SMEM, st>>>(a, am, bm);
  CB_CUDA(cudaGetLastError());
  dn::dense_reduce_kernel<<<(int)std::min<size_t>(((size_t)F * N / 4 + 255) / 256, 148 * 8), 256, 0, st>>>(partial, DENSE_KSPLIT, F, N, bias, out);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

int launch_dense_wgrad_tc(const Geom& g, const ParamMap& pm, int F, const bf16* A, const bf16* dy, float* grad, int* error_flag, cudaStream_t st) {
  if (F <= 0) return CB_OK;
  const int K = g.H * g.W * g.Cin, N = g.Cout;
  CUtensorMap am, bm;
  if (!map2d(&am, A, F, K) || !map2d(&bm, dy, F, N)) { set_error("cuTensorMapEncodeTiled refused a dense-layer map"); return CB_ECUDA; }
  dn::Args a{nullptr, nullptr, nullptr, nullptr, grad, F, K, N, g.H, g.W, g.Cin, pm.w_off, error_flag};
  int rc = ensure_dyn_smem((const void*)dn::dense_wgrad_kernel, dn::SMEM); if (rc) return rc;
  dn::dense_wgrad_kernel<<<dim3((K + dn::BM - 1) / dn::BM, (N + dn::BN - 1) / dn::BN), dn::NTHREADS, dn::SMEM, st>>>(a, am, bm);
  CB_CUDA(cudaGetLastError());
  dn::colsum_kernel<<<N / 8, 256, 0, st>>>(dy, F, N, grad + pm.b_off);      // N % 64 == 0 (dense_tc_supported)
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

// dgrad of the fc layer: dx [F][K] = gate(dY [F][N] . Wf^T), gated by the sign of the stored feature map
int launch_dense_dgrad_tc(const Geom& g, int F, const bf16* dy, const bf16* wf, const bf16* mask, bf16* dx, int* error_flag, cudaStream_t st) {
  if (F <= 0) return CB_OK;
  const int K = g.H * g.W * g.Cin, N = g.Cout;
  CUtensorMap am, bm;
  if (!map2d(&am, dy, F, N) || !map2d(&bm, wf, K, N)) { set_error("cuTensorMapEncodeTiled refused a dense-layer map"); return CB_ECUDA; }
  dn::Args a{nullptr, mask, dx, nullptr, nullptr, F, K, N, g.H, g.W, g.Cin, 0, error_flag};
  int rc = ensure_dyn_smem((const void*)dn::dense_kmajor_kernel<2>, dn::SMEM2); if (rc) return rc;
  dn::dense_kmajor_kernel<2><<<dim3((F + dn::BM - 1) / dn::BM, (K + dn::BN - 1) / dn::BN, 1), dn::NTHREADS, dn::SMEM2, st>>>(a, am, bm);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

}  // namespace cb
