// tcgen05 / TMEM implicit-GEMM 3x3 convolution (stride 1, zero pad 1) for CB_PREC_BF16_TC, sm_100a.
//
// One kernel serves the forward conv and its dgrad (the same convolution with flipped taps and
// transposed weights; only the packed weights and the epilogue differ).
//
// Data layout in shared memory ("pixel-linear planes"): a group of G frames is staged with its zero
// halo as  plane[c/8][j*R + (y+1)*Wp + (x+1)][c%8],  R = (H+2)*(W+2), Wp = W+2, 16 bytes per (pixel,
// channel-chunk).  For an output position q = j*R + y*Wp + x the input under tap (di,dj) is at the
// linear position q + di*Wp + dj: a tap is a constant shift of the start address.  A 128-row A operand
// (128 consecutive linear positions, 16 channels) is therefore exactly the canonical K-major
// no-swizzle UMMA layout (core matrix = 8 pixels x 16 B, SBO = 128 B, LBO = plane stride) for ANY tap,
// and the whole 3x3 conv is 9*Cin/16 tcgen05.mma instructions per 128-position tile with the fp32
// accumulator resident in TMEM.  Positions that fall on halo columns/rows are computed and dropped
// (6-40% of the rows, the price of needing no im2col and no per-tap copies).
// Weights: B operand [Cout x 16] per (tap, k-step), K-major canonical layout, staged once per CTA.
#include "common.cuh"
#include "tma.cuh"

#include <cstring>

namespace cb {

namespace tc {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// UMMA shared-memory matrix descriptor, no swizzle (layout_type 0), version 1 (Blackwell)
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  uint64_t d = (uint64_t)((saddr >> 4) & 0x3FFFu);
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFFu) << 16;
  d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFFu) << 32;
  d |= (uint64_t)1 << 46;
  return d;
}
// instruction descriptor, kind::f16: D fp32, A/B bf16; a_major/b_major: 0 = K-major, 1 = MN-major
__host__ __device__ constexpr uint32_t make_idesc(int M, int N, int a_mn, int b_mn) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)a_mn << 15) | ((uint32_t)b_mn << 16) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
__device__ __forceinline__ void mma_f16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}\n"
               :: "r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
// one lane of a converged warp: tcgen05 instructions then issue from the uniform datapath (see tc_ptx.cuh)
__device__ __forceinline__ bool elect_one() {
  uint32_t pred = 0;
  asm volatile("{\n\t.reg .b32 rx;\n\t.reg .pred px;\n\telect.sync rx|px, %1;\n\t@px mov.s32 %0, 1;\n\t}\n" : "+r"(pred) : "r"(0xFFFFFFFFu));
  return pred != 0;
}
__device__ __forceinline__ void mma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n" :: "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" :: "r"(bar), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
}
// bounded spin: a descriptor mistake must not hang the GPU box; returns false on timeout
__device__ __forceinline__ bool mbar_wait(uint32_t bar, uint32_t parity) {
  for (uint32_t it = 0; it < (1u << 24); ++it) {
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    if (ok) return true;
  }
  return false;
}
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory"); }
__device__ __forceinline__ void tmem_alloc(uint32_t dst_smem, uint32_t cols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" :: "r"(dst_smem), "r"(cols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t cols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" :: "r"(taddr), "r"(cols) : "memory");
}
// 16 consecutive fp32 columns of this thread's TMEM lane
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float* v) {
  uint32_t r[16];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];\n"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
                 "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
               : "r"(taddr) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}

struct ConvTcArgs {
  const bf16* in;      // [F, H, W, CIN]
  const bf16* w;       // packed B operand: [tap][CIN/8][COUT][8]
  const float* bias;   // [COUT] (forward) or nullptr
  const bf16* aux0;    // forward: skip tensor (added) | dgrad: pre-activation whose sign gates the result; nullable
  const bf16* aux1;    // dgrad: gradient added after gating; nullable
  bf16* out;           // [F, H, W, COUT]
  int F, H, W, G, npix_alloc, relu_in, use_tma, relu_out;
  int RB, nbands;      // rows per band (= H when the whole frame is staged) and bands per frame (banded: G = 1, TMA only)
  int* error_flag;
};

constexpr int TMEM_COLS = 128;     // 128 columns and <= 72 KB of shared memory per CTA: three CTAs per SM overlap their phases
constexpr int NT = 256;            // two warpgroups: both stage operands; each drains every second accumulator tile

// MODE 0: out = acc + bias (+ aux0).   MODE 1: out = (aux0 ? (aux0 > 0 ? acc : 0) : acc) (+ aux1).
template <int CIN, int COUT, int MODE>
__global__ void __launch_bounds__(NT) conv3x3_tc_kernel(const ConvTcArgs a, const __grid_constant__ CUtensorMap tmap) {
  extern __shared__ __align__(128) uint8_t smem[];
  constexpr int NCH = CIN / 8, KSTEPS = CIN / 16, TILES_PER_BATCH = TMEM_COLS / COUT;
  constexpr uint32_t W_BYTES = 9u * CIN * COUT * 2u;
  __shared__ __align__(8) uint64_t bar_storage;
  __shared__ __align__(8) uint64_t ldbar_storage;
  __shared__ uint32_t tmem_base_smem;
  const int tid = threadIdx.x, warp = tid >> 5, wg = warp >> 2, lane_row = tid & 127;
  const int Wp = a.W + 2, R = (a.RB + 2) * Wp;      // R = staged positions per frame (band with its halo)
  uint8_t* w_smem = smem;
  uint8_t* in_smem = smem + ((W_BYTES + 127u) & ~127u);
  const uint32_t plane_bytes = (uint32_t)a.npix_alloc * 16u;
  const uint32_t bar = smem_u32(&bar_storage);

  const uint32_t ldbar = smem_u32(&ldbar_storage);
  if (tid == 0) { mbar_init(bar, 1); mbar_init(ldbar, 1); if (a.use_tma) tma::prefetch_map(&tmap); }
  if (warp == 0) tmem_alloc(smem_u32(&tmem_base_smem), TMEM_COLS);
  // weights (already in operand layout) and a zeroed input area (halo and slack stay zero for the whole kernel)
  for (uint32_t i = tid; i < W_BYTES / 16; i += NT) reinterpret_cast<uint4*>(w_smem)[i] = reinterpret_cast<const uint4*>(a.w)[i];
  for (uint32_t i = tid; i < plane_bytes * NCH / 16; i += NT) reinterpret_cast<uint4*>(in_smem)[i] = make_uint4(0, 0, 0, 0);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_smem;
  const uint32_t idesc = make_idesc(128, COUT, 0, 0);
  const uint32_t a_base = smem_u32(in_smem), b_base = smem_u32(w_smem);
  uint32_t parity = 0, ldparity = 0;
  const int ngroups = ((a.F + a.G - 1) / a.G) * a.nbands;

  for (int grp = blockIdx.x; grp < ngroups; grp += gridDim.x) {
    const int fg = grp / a.nbands, yb = (grp - fg * a.nbands) * a.RB;
    const int f0 = fg * a.G, nf = min(a.G, a.F - f0);
    // ---- stage the group's frames: global NHWC -> planes, ReLU on the way in --------------------------
    if (a.use_tma) {
      // ---- TMA: one bulk tensor copy per 8-channel chunk lands the whole group, zero halo included (box starts at (-1,-1)) ----
      const uint32_t bytes = (uint32_t)(a.G * R) * 16u;
      if (tid == 0) {
        tma::arrive_expect_tx(ldbar, bytes * NCH);
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) tma::load_4d(a_base + (uint32_t)ch * plane_bytes, &tmap, ch * 8, -1, yb - 1, f0, ldbar);
      }
      if (!mbar_wait(ldbar, ldparity)) { if (a.error_flag) *a.error_flag = 6; }
      ldparity ^= 1;
      if (a.relu_in) {      // ReLU in place (generic proxy), made visible to the tensor core by the proxy fence below
        const int n16 = a.G * R;
        for (int i = tid; i < n16 * NCH; i += NT) {
          const int ch = i / n16, pos = i - ch * n16;
          uint4* p = reinterpret_cast<uint4*>(in_smem + (size_t)ch * plane_bytes + (size_t)pos * 16);
          uint4 v = *p;
          __nv_bfloat162* h = reinterpret_cast<__nv_bfloat162*>(&v);
          const __nv_bfloat162 z = __float2bfloat162_rn(0.f);
#pragma unroll
          for (int k = 0; k < 4; ++k) h[k] = __hmax2(h[k], z);
          *p = v;
        }
      }
    } else {
    const int per_frame = a.H * a.W * NCH, nwork = a.G * per_frame;
    for (int i0 = tid; i0 < nwork; i0 += NT * 4) {       // 4 independent 16-byte loads in flight per thread
      uint4 v[4]; uint32_t dst[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int i = i0 + u * NT;
        v[u] = make_uint4(0, 0, 0, 0); dst[u] = 0xFFFFFFFFu;
        if (i < nwork) {
          int j = i / per_frame, rem = i - j * per_frame;
          int ch = rem % NCH, pix = rem / NCH;
          int y = pix / a.W, x = pix - y * a.W;
          dst[u] = (uint32_t)ch * plane_bytes + (uint32_t)(j * R + (y + 1) * Wp + (x + 1)) * 16u;
          if (j < nf) v[u] = *reinterpret_cast<const uint4*>(a.in + ((size_t)(f0 + j) * a.H * a.W + pix) * CIN + ch * 8);
        }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        if (dst[u] == 0xFFFFFFFFu) continue;
        if (a.relu_in) {
          __nv_bfloat162* h = reinterpret_cast<__nv_bfloat162*>(&v[u]);
          const __nv_bfloat162 z = __float2bfloat162_rn(0.f);
#pragma unroll
          for (int k = 0; k < 4; ++k) h[k] = __hmax2(h[k], z);
        }
        *reinterpret_cast<uint4*>(in_smem + dst[u]) = v[u];
      }
    }
    }
    fence_async_smem();
    __syncthreads();
    const int ntiles = ((nf - 1) * R + a.RB * Wp + 127) / 128;      // positions up to the last computed row of the last frame
    for (int t0 = 0; t0 < ntiles; t0 += TILES_PER_BATCH) {
      const int nt = min(TILES_PER_BATCH, ntiles - t0);
      if (tid < 32) {        // the whole warp runs the loop, one elected lane issues
        tc_fence_after();
        const uint32_t a_lo = ((a_base >> 4) & 0x3FFFu) | (((plane_bytes >> 4) & 0x3FFFu) << 16), d_hi = 8u | (1u << 14);   // LBO = plane, SBO = 128 B
        const uint32_t b_lo = ((b_base >> 4) & 0x3FFFu) | ((uint32_t)COUT << 16);                                        // LBO = COUT*16 B
        for (int s = 0; s < nt; ++s) {
          const uint32_t q0 = (uint32_t)(t0 + s) * 128u;
#pragma unroll
          for (int tap = 0; tap < 9; ++tap) {
            const uint32_t shift = (uint32_t)((tap / 3) * Wp + (tap % 3));
#pragma unroll
            for (int ks = 0; ks < KSTEPS; ++ks) {
              const uint64_t ad = ((uint64_t)d_hi << 32) | (uint64_t)(a_lo + q0 + shift + (uint32_t)(2 * ks) * (plane_bytes >> 4));
              const uint64_t bd = ((uint64_t)d_hi << 32) | (uint64_t)(b_lo + (uint32_t)((tap * NCH + 2 * ks) * COUT));
              if (elect_one()) mma_f16(tmem_base + (uint32_t)(s * COUT), ad, bd, idesc, (tap | ks) ? 1u : 0u);
            }
          }
        }
        if (elect_one()) mma_commit(bar);
        __syncwarp();
      }
      if (!mbar_wait(bar, parity)) { if (a.error_flag) *a.error_flag = 1; }
      parity ^= 1;
      tc_fence_after();
      // ---- epilogue: TMEM lane = tile row = linear position; one thread per position ----------------------
      for (int s = wg; s < nt; s += 2) {
        const int q = (t0 + s) * 128 + lane_row;
        const int j = q / R, rem = q - j * R;
        const int yl = rem / Wp, x = rem - yl * Wp, y = yb + yl;
        const bool valid = j < nf && yl < a.RB && y < a.H && x < a.W;
        const size_t o = (((size_t)(f0 + j) * a.H + y) * a.W + x) * COUT;
#pragma unroll
        for (int c0 = 0; c0 < COUT; c0 += 16) {
          float v[16];
          tmem_ld16(tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)(s * COUT + c0), v);   // warp-collective: no divergence before it
          if (!valid) continue;
          if (MODE == 0) {
#pragma unroll
            for (int i = 0; i < 16; ++i) v[i] += a.bias[c0 + i];
            if (a.aux0) {
              uint4 s0 = *reinterpret_cast<const uint4*>(a.aux0 + o + c0), s1 = *reinterpret_cast<const uint4*>(a.aux0 + o + c0 + 8);
              const bf16* h0 = reinterpret_cast<const bf16*>(&s0); const bf16* h1 = reinterpret_cast<const bf16*>(&s1);
#pragma unroll
              for (int i = 0; i < 8; ++i) { v[i] += __bfloat162float(h0[i]); v[8 + i] += __bfloat162float(h1[i]); }
            }
            if (a.relu_out) {
#pragma unroll
              for (int i = 0; i < 16; ++i) v[i] = fmaxf(v[i], 0.f);
            }
          } else {
            if (a.aux0) {
              uint4 s0 = *reinterpret_cast<const uint4*>(a.aux0 + o + c0), s1 = *reinterpret_cast<const uint4*>(a.aux0 + o + c0 + 8);
              const bf16* h0 = reinterpret_cast<const bf16*>(&s0); const bf16* h1 = reinterpret_cast<const bf16*>(&s1);
#pragma unroll
              for (int i = 0; i < 8; ++i) { if (!(__bfloat162float(h0[i]) > 0.f)) v[i] = 0.f; if (!(__bfloat162float(h1[i]) > 0.f)) v[8 + i] = 0.f; }
            }
            if (a.aux1) {
              uint4 s0 = *reinterpret_cast<const uint4*>(a.aux1 + o + c0), s1 = *reinterpret_cast<const uint4*>(a.aux1 + o + c0 + 8);
              const bf16* h0 = reinterpret_cast<const bf16*>(&s0); const bf16* h1 = reinterpret_cast<const bf16*>(&s1);
#pragma unroll
              for (int i = 0; i < 8; ++i) { v[i] += __bfloat162float(h0[i]); v[8 + i] += __bfloat162float(h1[i]); }
            }
          }
          uint4 o0, o1;
          __nv_bfloat162* p0 = reinterpret_cast<__nv_bfloat162*>(&o0); __nv_bfloat162* p1 = reinterpret_cast<__nv_bfloat162*>(&o1);
#pragma unroll
          for (int i = 0; i < 4; ++i) { p0[i] = __floats2bfloat162_rn(v[2 * i], v[2 * i + 1]); p1[i] = __floats2bfloat162_rn(v[8 + 2 * i], v[8 + 2 * i + 1]); }
          *reinterpret_cast<uint4*>(a.out + o + c0) = o0;
          *reinterpret_cast<uint4*>(a.out + o + c0 + 8) = o1;
        }
      }
      tc_fence_before();
      __syncthreads();      // TMEM drained and (after the last batch) the staged frames free for the next group
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem_base, TMEM_COLS);
}

}  // namespace tc

// ---- host side ---------------------------------------------------------------------------------
bool conv_tc_supported(const Geom& g) {
  auto okc = [](int c) { return c == 16 || c == 32 || c == 64; };
  return g.kh == 3 && g.kw == 3 && g.s == 1 && g.p == 1 && okc(g.Cin) && okc(g.Cout) && g.H == g.Ho && g.W == g.Wo;
}

struct TcPlan { int G, npix_alloc, RB, nbands; size_t smem; };
static TcPlan tc_plan(int H, int W, int cin, int cout) {
  const int Wp = W + 2, R = (H + 2) * Wp;
  const size_t wbytes = ((size_t)9 * cin * cout * 2 + 127) & ~(size_t)127;
  // shared-memory target per CTA: three CTAs per SM (72 KB) unless the weight image alone is large (two CTAs, 110 KB);
  // co-resident CTAs overlap each other's staging / MMA / epilogue phases
  const size_t budget = wbytes <= 40 * 1024 ? 72 * 1024 : 110 * 1024;
  auto alloc_pix = [&](int positions) { int n = ((positions + 127) / 128) * 128 + 2 * Wp + 2; return (n + 7) / 8 * 8; };
  TcPlan p;
  p.G = (int)((budget - wbytes) / ((size_t)R * cin * 2)); if (p.G > 8) p.G = 8;
  p.RB = H; p.nbands = 1;
  while (p.G > 1 && wbytes + (size_t)alloc_pix(p.G * R) * cin * 2 > budget) --p.G;
  if (p.G < 1 || wbytes + (size_t)alloc_pix(p.G * R) * cin * 2 > budget) {
    p.G = 1;
    if (wbytes + (size_t)alloc_pix(R) * cin * 2 > budget) {      // one frame is too big: row bands of RB rows (+2 halo rows)
      long rows = ((long)(budget - wbytes) / ((long)cin * 2) - 2 * Wp - 140) / Wp - 2;
      if (rows < 4) rows = 4;
      p.nbands = (int)((H + rows - 1) / rows); p.RB = (H + p.nbands - 1) / p.nbands;
    }
  }
  p.npix_alloc = alloc_pix(p.nbands > 1 ? (p.RB + 2) * Wp : p.G * R);
  p.smem = wbytes + (size_t)p.npix_alloc * cin * 2;
  return p;
}

// the staged frame group (with halo) plus the weight image must fit one CTA's shared memory
bool conv_tc_fits(int H, int W, int cin, int cout) { return tc_plan(H, W, cin, cout).smem <= 220 * 1024; }

template <int CIN, int COUT, int MODE>
static int launch_one(const tc::ConvTcArgs& a, const CUtensorMap& tmap, size_t smem, int ngroups, cudaStream_t st) {
  static size_t configured = 0;      // largest dynamic size this instantiation has been opted in for
  if (smem > configured) {
    CB_CUDA(cudaFuncSetAttribute(tc::conv3x3_tc_kernel<CIN, COUT, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    configured = smem;
  }
  int grid = std::min(ngroups, 3 * 148);
  tc::conv3x3_tc_kernel<CIN, COUT, MODE><<<grid, tc::NT, smem, st>>>(a, tmap);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

template <int MODE>
static int dispatch(int cin, int cout, const tc::ConvTcArgs& a, const CUtensorMap& tmap, size_t smem, int ngroups, cudaStream_t st) {
#define CB_TC_CASE(ci, co) if (cin == ci && cout == co) return launch_one<ci, co, MODE>(a, tmap, smem, ngroups, st);
  CB_TC_CASE(16, 16) CB_TC_CASE(16, 32) CB_TC_CASE(32, 16) CB_TC_CASE(32, 32) CB_TC_CASE(32, 64) CB_TC_CASE(64, 32) CB_TC_CASE(64, 64)
  CB_TC_CASE(16, 64) CB_TC_CASE(64, 16)
#undef CB_TC_CASE
  set_error("conv_tc: unsupported channel counts %d -> %d", cin, cout);
  return CB_EINVAL;
}

// mode 0: forward (cin = g.Cin, cout = g.Cout);  mode 1: dgrad (cin = g.Cout, cout = g.Cin, weights packed flipped/transposed)
int launch_conv_tc(int mode, int F, int H, int W, int cin, int cout, const bf16* in, const bf16* w, const float* bias, const bf16* aux0,
                   const bf16* aux1, bf16* out, bool relu_in, bool relu_out, int* error_flag, cudaStream_t st) {
  if (F <= 0) return CB_OK;
  TcPlan p = tc_plan(H, W, cin, cout);
  if (p.smem > 220 * 1024) { set_error("conv_tc: frame does not fit shared memory"); return CB_EINVAL; }
  CUtensorMap tmap; memset(&tmap, 0, sizeof tmap);
  const bool use_tma = W + 2 <= 256 && p.RB + 2 <= 256 && tma::make_nhwc_map(&tmap, in, F, H, W, cin, W + 2, p.RB + 2, p.G);
  if (!use_tma && p.nbands > 1) { set_error("conv_tc: banded staging needs TMA"); return CB_EINVAL; }
  tc::ConvTcArgs a{in, w, bias, aux0, aux1, out, F, H, W, p.G, p.npix_alloc, relu_in ? 1 : 0, use_tma ? 1 : 0, relu_out ? 1 : 0, p.RB, p.nbands, error_flag};
  int ngroups = ((F + p.G - 1) / p.G) * p.nbands;
  return mode == 0 ? dispatch<0>(cin, cout, a, tmap, p.smem, ngroups, st) : dispatch<1>(cin, cout, a, tmap, p.smem, ngroups, st);
}

}  // namespace cb
