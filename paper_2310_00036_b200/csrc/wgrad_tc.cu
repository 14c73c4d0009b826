// tcgen05 / TMEM weight-gradient kernel for 3x3 stride-1 pad-1 convolutions, CB_PREC_BF16_TC, sm_100a.
//
//   dW[tap][c][o] = sum_q X[q + shift(tap)][c] * DY[q][o]        db[o] = sum_q DY[q][o]
//
// with q running over the pixel-linear positions of conv_tc.cu (DY is staged with zeros at halo
// positions, X with its zero halo and ReLU applied on the way in).  The contraction index is the PIXEL, so
// both operands are MN-major: in the plane layout plane[ch/8][q][ch%8] (16 B per (position, chunk)) a
// core matrix is 8 positions x 8 channels with the K rows 16 B apart -- exactly the canonical MN-major
// no-swizzle UMMA layout (LBO = 128 B between groups of 8 positions, SBO = plane stride between groups
// of 8 channels).  A tap is again a constant shift of A's start address.
//
// UMMA needs M = 128 rows while a layer has Cin = 16/32 (+1 bias row) real ones: the descriptor simply
// walks on into the following planes (a plane of ones for the bias row, then DY, then zeros); those
// rows of D are never read.  The 9 accumulators [128 x Cout] stay in TMEM (9*Cout <= 288 columns) for
// the whole life of the CTA, which runs over a fixed set of (frame-group, row-band) work items and
// writes ONE fp32 partial [9][Cin+1][Cout] at the end; a second kernel adds the partials in CTA order,
// so the result is bitwise reproducible (no atomics; the item -> CTA map depends on the shape only).
#include "common.cuh"
#include "tma.cuh"

#include <cstring>

namespace cb {
namespace tcw {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  uint64_t d = (uint64_t)((saddr >> 4) & 0x3FFFu);
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFFu) << 16;
  d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFFu) << 32;
  d |= (uint64_t)1 << 46;
  return d;
}
__device__ __forceinline__ void mma_f16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}\n"
               :: "r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
// one lane of a converged warp; the compiler then issues the tcgen05 instruction from the uniform datapath
// instead of looping over the active lanes of a divergent branch (which costs ~50 clk per MMA)
__device__ __forceinline__ bool elect_one() {
  uint32_t pred = 0;
  asm volatile("{\n\t.reg .b32 rx;\n\t.reg .pred px;\n\telect.sync rx|px, %1;\n\t@px mov.s32 %0, 1;\n\t}\n" : "+r"(pred) : "r"(0xFFFFFFFFu));
  return pred != 0;
}
__device__ __forceinline__ void mma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n" :: "r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_wait(uint32_t bar, uint32_t parity) {
  for (uint32_t it = 0; it < (1u << 24); ++it) {
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    if (ok) return true;
  }
  return false;
}
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

struct WgradTcArgs {
  const bf16* x;      // [F, H, W, CIN]  layer input (pre-activation when relu_in)
  const bf16* dy;     // [F, H, W, COUT]
  float* partial;     // [gridDim.x][9][CIN+1][COUT]
  int F, H, W, G, R, nbands, npix_alloc, kext, relu_in, stage_planes, use_tma, dy_rows;
  int repl;           // ST3 with TMA: only the dj = 0 planes are landed (the TMA unit moves about one 16-byte piece per clock, so three
                      // shifted boxes would bound the kernel); the loader warps derive the dj = 1, 2 copies in shared memory
  int c_off, cin_total;      // the kernel handles input channels [c_off, c_off + CIN) of a layer with cin_total channels
  int* error_flag;
};

__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}\n" :: "r"(bar) : "memory");
}

constexpr int NLOAD = 256;       // warps 0-7: stage operands (warps 0-3 later read TMEM); warp 8: one thread issues the MMAs

// UM = UMMA M (64 or 128): rows 0..CIN(+bias) are real, the rest walks into the following planes and is ignored.
// Two shared-memory stages: the loader warps fill stage s+1 while the tensor core works on stage s.
// ST3 (Cin = 16 only): the loaders store every X element three times, shifted by dj = 0,1,2 positions, into planes
// (dj, chunk); the M walk of ONE MMA then covers the three taps (di, 0..2) at rows dj*CIN + c -- 3 instead of 9
// MMAs per 16 positions, and 49 instead of 17 useful rows of 64.
template <int CIN, int COUT, int UM, bool ST3>
__global__ void __launch_bounds__(NLOAD + 64) wgrad3x3_tc_kernel(const WgradTcArgs a, const __grid_constant__ CUtensorMap xmap, const __grid_constant__ CUtensorMap ymap) {
  extern __shared__ __align__(128) uint8_t smem[];
  constexpr int XCH = CIN / 8, YCH = COUT / 8, XPL = ST3 ? 3 * XCH : XCH;      // X planes per stage
  constexpr int NACC = ST3 ? 3 : 9;
  constexpr uint32_t TCOLS = (NACC * COUT <= 128) ? 128u : ((NACC * COUT <= 256) ? 256u : 512u);
  static_assert(!ST3 || 3 * CIN + 1 <= UM, "3-tap stacking needs 3*CIN+1 rows");
  __shared__ __align__(8) uint64_t bars[7];          // full[2], empty[2], done, raw[2] (TMA landed)
  __shared__ uint32_t tmem_base_smem;
  const int tid = threadIdx.x, warp = tid >> 5;
  const int Wp = a.W + 2, Rb = (a.R + 2) * Wp;          // positions per frame region of a band
  const uint32_t P = (uint32_t)a.npix_alloc * 16u;      // plane stride
  const uint32_t stage_bytes = (uint32_t)a.stage_planes * P;
  // per stage: planes [0, XCH) X | XCH: ones (bias row) | [XCH+1, XCH+1+YCH) DY | padding planes (zeros)
  const uint32_t bar0 = smem_u32(&bars[0]);
  if (tid == 0) {
    for (int i = 0; i < 7; ++i) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" :: "r"(bar0 + 8u * i) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  if (warp == NLOAD / 32) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" :: "r"(smem_u32(&tmem_base_smem)), "r"(TCOLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
  }
  // total allocation: the last stage's A descriptor may walk UM/8 planes from its start
  const uint32_t total_bytes = stage_bytes + (uint32_t)max(a.stage_planes, UM / 8) * P;
  for (uint32_t i = tid; i < total_bytes / 16; i += NLOAD + 64) reinterpret_cast<uint4*>(smem)[i] = make_uint4(0, 0, 0, 0);
  __syncthreads();
  {
    const uint32_t one2 = 0x3F803F80u;    // two bf16 ones
    for (int st = 0; st < 2; ++st)
      for (uint32_t i = tid; i < P / 16; i += NLOAD + 64) reinterpret_cast<uint4*>(smem + (size_t)st * stage_bytes + (size_t)XPL * P)[i] = make_uint4(one2, one2, one2, one2);
  }
  asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
  const uint32_t tmem_base = tmem_base_smem;
  const int ngroups = (a.F + a.G - 1) / a.G, nitems = ngroups * a.nbands;
  const int my_items = ((int)blockIdx.x < nitems) ? (nitems - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;

  const bool direct = a.use_tma && !a.relu_in && !a.repl;      // nothing to do between the TMA landing and the MMAs: the issuer waits on raw[] itself
  if (warp < NLOAD / 32) {
    // ================= loaders =================
    for (int it = 0; it < (direct ? 0 : my_items); ++it) {
      const int item = blockIdx.x + it * gridDim.x, s = it & 1, use = it >> 1;
      if (!a.use_tma && use > 0 && !mbar_wait(bar0 + 8u * (2 + s), (uint32_t)((use - 1) & 1))) { if (a.error_flag) *a.error_flag = 2; }
      uint8_t* xs = smem + (size_t)s * stage_bytes;
      uint8_t* ys = xs + (size_t)(XPL + 1) * P;
      const int grp = item / a.nbands, band = item - grp * a.nbands;
      const int f0 = grp * a.G, nf = min(a.G, a.F - f0), yb = band * a.R;
      if (a.use_tma) {
        // operands were landed by the TMA producer thread; only the ReLU (in place) is left to these warps
        if (!mbar_wait(bar0 + 8u * (5 + s), (uint32_t)(use & 1))) { if (a.error_flag) *a.error_flag = 7; }
        if (a.repl) {
          const int n16 = a.G * Rb;
          const __nv_bfloat162 z = __float2bfloat162_rn(0.f);
          for (int i = tid; i < n16 * XCH; i += NLOAD) {
            const int ch = i / n16, pos = i - ch * n16;
            uint8_t* p = xs + (size_t)ch * P + (size_t)pos * 16;
            uint4 v = *reinterpret_cast<uint4*>(p);
            if (a.relu_in) {
              __nv_bfloat162* h = reinterpret_cast<__nv_bfloat162*>(&v);
#pragma unroll
              for (int k = 0; k < 4; ++k) h[k] = __hmax2(h[k], z);
              *reinterpret_cast<uint4*>(p) = v;
            }
            if (pos >= 1) *reinterpret_cast<uint4*>(p + (size_t)XCH * P - 16) = v;          // plane (1, ch), one position earlier
            if (pos >= 2) *reinterpret_cast<uint4*>(p + (size_t)2 * XCH * P - 32) = v;      // plane (2, ch), two positions earlier
          }
        } else if (a.relu_in) {
          const int n16 = a.G * Rb;
          for (int i = tid; i < n16 * XPL; i += NLOAD) {
            const int pl = i / n16, pos = i - pl * n16;
            uint4* p = reinterpret_cast<uint4*>(xs + (size_t)pl * P + (size_t)pos * 16);
            uint4 v = *p;
            __nv_bfloat162* h = reinterpret_cast<__nv_bfloat162*>(&v);
            const __nv_bfloat162 z = __float2bfloat162_rn(0.f);
#pragma unroll
            for (int k = 0; k < 4; ++k) h[k] = __hmax2(h[k], z);
            *p = v;
          }
        }
      } else {
      const int xn = a.G * Rb * XCH;
      for (int i0 = tid; i0 < xn; i0 += NLOAD * 4) {
        uint4 v[4]; uint32_t dst[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int i = i0 + u * NLOAD;
          v[u] = make_uint4(0, 0, 0, 0); dst[u] = 0xFFFFFFFFu;
          if (i < xn) {
            int ch = i % XCH, pos = i / XCH;
            int j = pos / Rb, rem = pos - j * Rb, lr = rem / Wp, xp = rem - lr * Wp;
            int y = yb - 1 + lr, x = xp - 1;
            dst[u] = (uint32_t)ch * P + (uint32_t)pos * 16u;
            if (j < nf && (unsigned)y < (unsigned)a.H && (unsigned)x < (unsigned)a.W)
              v[u] = *reinterpret_cast<const uint4*>(a.x + (((size_t)(f0 + j) * a.H + y) * a.W + x) * a.cin_total + a.c_off + ch * 8);
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
          *reinterpret_cast<uint4*>(xs + dst[u]) = v[u];
          if (ST3) {      // dst = ch*P + pos*16: the copies for dj = 1, 2 live XCH / 2*XCH planes further, 1 / 2 positions earlier
            const uint32_t pos16 = dst[u] % P;
            if (pos16 >= 16u) *reinterpret_cast<uint4*>(xs + dst[u] + (uint32_t)XCH * P - 16u) = v[u];
            if (pos16 >= 32u) *reinterpret_cast<uint4*>(xs + dst[u] + 2u * (uint32_t)XCH * P - 32u) = v[u];
          }
        }
      }
      const int yn = a.kext * YCH;
      for (int i0 = tid; i0 < yn; i0 += NLOAD * 4) {
        uint4 v[4]; uint32_t dst[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int i = i0 + u * NLOAD;
          v[u] = make_uint4(0, 0, 0, 0); dst[u] = 0xFFFFFFFFu;
          if (i < yn) {
            int ch = i % YCH, pos = i / YCH;
            int j = pos / Rb, rem = pos - j * Rb, lr = rem / Wp, x = rem - lr * Wp;
            int y = yb + lr;
            dst[u] = (uint32_t)ch * P + (uint32_t)pos * 16u;
            if (j < nf && lr < a.R && y < a.H && x < a.W)
              v[u] = *reinterpret_cast<const uint4*>(a.dy + (((size_t)(f0 + j) * a.H + y) * a.W + x) * COUT + ch * 8);
          }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) if (dst[u] != 0xFFFFFFFFu) *reinterpret_cast<uint4*>(ys + dst[u]) = v[u];
      }
      }
      asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
      asm volatile("bar.sync 1, %0;\n" :: "n"(NLOAD) : "memory");
      if (tid == 0) mbar_arrive(bar0 + 8u * s);
    }
    // ================= epilogue (warps 0-3 own the TMEM lanes) =================
    if (warp < 4) {
    if (my_items > 0 && !mbar_wait(bar0 + 8u * 4, 0u)) { if (a.error_flag) *a.error_flag = 2; }
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
    float* out = a.partial + (size_t)blockIdx.x * 9 * (CIN + 1) * COUT;
    // UM = 128: accumulator row r sits in TMEM lane r; UM = 64: in lane 32*(r/16) + r%16
    const int lane = tid & 31;
    const int row = (UM == 128) ? tid : ((lane < 16) ? warp * 16 + lane : 1 << 20);
    constexpr int LAST_ROW = ST3 ? 3 * CIN : CIN;         // the bias row
    const bool warp_needed = (UM == 128) ? (warp * 32 <= LAST_ROW) : (warp * 16 <= LAST_ROW);
    if (warp_needed) {
      for (int acc = 0; acc < NACC; ++acc) {
#pragma unroll
        for (int c0 = 0; c0 < COUT; c0 += 16) {
          float v[16];
          tmem_ld16(tmem_base + ((uint32_t)(warp * 32) << 16) + (uint32_t)(acc * COUT + c0), v);
          if (row > LAST_ROW) continue;
          int tap, r;
          if (ST3) { if (row == LAST_ROW) { if (acc) continue; tap = 0; r = CIN; } else { tap = acc * 3 + row / CIN; r = row % CIN; } }
          else { tap = acc; r = row; }
#pragma unroll
          for (int i = 0; i < 16; ++i) out[((size_t)tap * (CIN + 1) + r) * COUT + c0 + i] = v[i];
        }
      }
    }
    }
  } else if (tid == NLOAD + 32) {
    // ================= TMA producer: runs one stage ahead of the tensor core =================
    if (a.use_tma) {
      tma::prefetch_map(&xmap); tma::prefetch_map(&ymap);
      const uint32_t xbytes = (uint32_t)(a.G * Rb) * 16u, ybytes = (uint32_t)(a.G * a.dy_rows * Wp) * 16u;
      for (int it = 0; it < my_items; ++it) {
        const int item = blockIdx.x + it * gridDim.x, s = it & 1, use = it >> 1;
        if (use > 0 && !mbar_wait(bar0 + 8u * (2 + s), (uint32_t)((use - 1) & 1))) { if (a.error_flag) *a.error_flag = 7; }
        const int grp = item / a.nbands, band = item - grp * a.nbands, f0 = grp * a.G, yb = band * a.R;
        const uint32_t xs = smem_u32(smem + (size_t)s * stage_bytes), ys = xs + (uint32_t)(XPL + 1) * P, rb = bar0 + 8u * (5 + s);
        const int npl = a.repl ? XCH : XPL;
        tma::arrive_expect_tx(rb, xbytes * (uint32_t)npl + ybytes * YCH);
        for (int pl = 0; pl < npl; ++pl) {       // plane (dj, ch): X shifted by dj positions = box started dj columns further right
          const int dj = ST3 ? pl / XCH : 0, ch = ST3 ? pl % XCH : pl;
          tma::load_4d(xs + (uint32_t)pl * P, &xmap, a.c_off + ch * 8, -1 + dj, yb - 1, f0, rb);
        }
        for (int ch = 0; ch < YCH; ++ch) tma::load_4d(ys + (uint32_t)ch * P, &ymap, ch * 8, 0, yb, f0, rb);
      }
    }
  } else if (warp == NLOAD / 32) {
    // ================= MMA issuer: the whole warp runs the loop, one elected lane issues =================
    const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | (1u << 15) | (1u << 16) | ((uint32_t)(COUT >> 3) << 17) | ((uint32_t)(UM >> 4) << 24);
    const uint32_t desc_hi = ((P >> 4) & 0x3FFFu) | (1u << 14);        // SBO = plane stride, descriptor version bit 46
    uint32_t accumulate = 0;
    for (int it = 0; it < my_items; ++it) {
      const int s = it & 1, use = it >> 1;
      if (!mbar_wait(bar0 + 8u * (direct ? 5 + s : s), (uint32_t)(use & 1))) { if (a.error_flag) *a.error_flag = 2; }
      asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
      const uint32_t x_base = smem_u32(smem + (size_t)s * stage_bytes), y_base = x_base + (uint32_t)(XPL + 1) * P;
      const uint32_t x_lo = ((x_base >> 4) & 0x3FFFu) | (8u << 16), y_lo = ((y_base >> 4) & 0x3FFFu) | (8u << 16);   // LBO = 128 B
      for (int k0 = 0; k0 < a.kext; k0 += 16) {
        const uint64_t bd = ((uint64_t)desc_hi << 32) | (uint64_t)(y_lo + (uint32_t)k0);
#pragma unroll
        for (int acc = 0; acc < NACC; ++acc) {
          const uint32_t shift = ST3 ? (uint32_t)(acc * Wp) : (uint32_t)((acc / 3) * Wp + (acc % 3));
          const uint64_t ad = ((uint64_t)desc_hi << 32) | (uint64_t)(x_lo + (uint32_t)k0 + shift);
          if (elect_one()) mma_f16(tmem_base + (uint32_t)(acc * COUT), ad, bd, idesc, accumulate);
        }
        accumulate = 1;
      }
      if (elect_one()) mma_commit(bar0 + 8u * (2 + s));          // stage s may be refilled once these MMAs have read it
      __syncwarp();
    }
    if (elect_one()) mma_commit(bar0 + 8u * 4);                  // everything issued so far has completed -> accumulators final
    __syncwarp();
  }
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  if (warp == NLOAD / 32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" :: "r"(tmem_base), "r"(TCOLS) : "memory");
}

// sums the per-CTA partials in CTA order and scatters to the canonical gradient
// RL lanes per element: lane k adds the partials of CTAs [k*q, (k+1)*q) in order, then the RL sums are added in lane
// order -- a fixed association, so the result is reproducible, with 1/RL of the dependent-load latency.
constexpr int RL = 16;
__global__ void wgrad_tc_reduce_kernel(const float* __restrict__ partial, int nctas, Geom g, ParamMap pm, int cin_k, int c_off, float* __restrict__ grad) {
  const int rows = cin_k + 1, per = 9 * rows * g.Cout;      // cin_k = channels handled by the kernel launch that wrote `partial`
  const int t = blockIdx.x * blockDim.x + threadIdx.x, i = t / RL, part = t % RL;
  const int q = (nctas + RL - 1) / RL, z0 = part * q, z1 = min(nctas, z0 + q);
  float s = 0.f;
  if (i < per) {
    int z = z0;
    for (; z + 10 <= z1; z += 10) {      // 10 loads in flight (148 CTAs / 16 lanes), then the additions in CTA order
      float v[10];
#pragma unroll
      for (int k = 0; k < 10; ++k) v[k] = __ldg(partial + (size_t)(z + k) * per + i);
#pragma unroll
      for (int k = 0; k < 10; ++k) s += v[k];
    }
    for (; z < z1; ++z) s += partial[(size_t)z * per + i];
  }
  float tot = s;
#pragma unroll
  for (int k = 1; k < RL; ++k) tot += __shfl_down_sync(0xffffffffu, s, k);      // lane `part == 0` collects s_0 + s_1 + ... in order
  if (part != 0 || i >= per) return;
  int o = i % g.Cout, qq = i / g.Cout, row = qq % rows, tap = qq / rows;
  if (row == cin_k) { if (tap == 0 && c_off == 0) grad[pm.b(o)] = tot; return; }
  grad[pm.w(o, c_off + row, tap / 3, tap % 3, g)] = tot;
}

// the same reduction for a batch of layers: block b belongs to the job with first_block <= b < next first_block.  A block
// sums RB consecutive elements: warp `part` adds the partials of CTAs [part*q, (part+1)*q) in order (one 128-byte run per
// step), then thread (0, e) adds the RL sums in part order -- the association of wgrad_tc_reduce_kernel.
constexpr int RB = 32;
__global__ void __launch_bounds__(RL * RB) wgrad_tc_reduce_batch_kernel(const __grid_constant__ WgradReduceBatch b, float* __restrict__ grad) {
  __shared__ float sums[RL][RB];
  int j = 0;
  while (j + 1 < b.n && (int)blockIdx.x >= b.job[j + 1].first_block) ++j;
  const WgradReduceJob& q = b.job[j];
  const Geom g = q.g;
  const int cin_k = q.cin_k, nctas = q.nctas, rows = cin_k + 1, per = 9 * rows * g.Cout;
  const int part = threadIdx.x / RB, e = threadIdx.x % RB, i = ((int)blockIdx.x - q.first_block) * RB + e;
  const int qn = (nctas + RL - 1) / RL, z0 = part * qn, z1 = min(nctas, z0 + qn);
  const float* __restrict__ partial = q.partial;
  float s = 0.f;
  if (i < per) {
    int z = z0;
    for (; z + 10 <= z1; z += 10) {      // 10 loads in flight (148 CTAs / 16 lanes), then the additions in CTA order
      float v[10];
#pragma unroll
      for (int k = 0; k < 10; ++k) v[k] = __ldg(partial + (size_t)(z + k) * per + i);
#pragma unroll
      for (int k = 0; k < 10; ++k) s += v[k];
    }
    for (; z < z1; ++z) s += partial[(size_t)z * per + i];
  }
  sums[part][e] = s;
  __syncthreads();
  if (part != 0 || i >= per) return;
  float tot = s;
#pragma unroll
  for (int k = 1; k < RL; ++k) tot += sums[k][e];
  int o = i % g.Cout, qq = i / g.Cout, row = qq % rows, tap = qq / rows;
  if (row == cin_k) { if (tap == 0 && q.c_off == 0) grad[q.pm.b(o)] = tot; return; }
  grad[q.pm.w(o, q.c_off + row, tap / 3, tap % 3, g)] = tot;
}

// ------------------------------------------------------------------------------------------------
// Swizzled variant (TMA, Cin in {16, 32}): whole pixels are landed once, one shared-memory row of 2*CIN (X) or 2*COUT (DY)
// bytes per position, in the 32B/64B/128B swizzle pattern.  The A descriptor is MN-major with LBO = one row: the M walk
// steps to the NEXT POSITION, so rows dj*CIN + c of one MMA are the taps (di, 0..2) without any shifted copy of X
// (the pattern is a function of the absolute address, so descriptors may start at any row).  The B descriptor walks N the
// same way with LBO = one image row: column group e of the MMA reads DY one row further down, which pairs it with the tap
// row di = 2 - e.  ONE MMA [UM x 3*COUT] per 16 positions therefore yields all nine taps; the accumulator stays in TMEM;
// the bias gradient is summed from the landed DY rows by the loader warps.
//   warps 0-7  wait for a landed stage, apply the ReLU in place when the layer needs it, add DY into the bias sums
//   warp 8     MMA issuer        warp 9  TMA producer (ring of `nstages` stages)
struct WgradSwArgs {
  float* partial; int F, H, W, G, R, nbands, npix_alloc, kext, relu_in, dy_rows, nstages;
  uint32_t stage_bytes, y_off;
  int dy_off;         // DY position p is stored at row p + dy_off (dy_off >= 2*(W+2), a multiple of the swizzle period)
  int x_off;          // X position p is stored at row p + x_off (>= 16: the first K step may start up to 15 rows early)
  int* error_flag;
};
constexpr int SW_MAX_STAGES = 3;

template <int CIN, int COUT>
__global__ void __launch_bounds__(NLOAD + 64) wgrad3x3_sw_kernel(const WgradSwArgs a, const __grid_constant__ CUtensorMap xmap, const __grid_constant__ CUtensorMap ymap) {
  extern __shared__ __align__(128) uint8_t smem_raw[];
  constexpr int UM = CIN == 16 ? 64 : 128;
  constexpr bool TWO = CIN == 64;      // 3*CIN = 192 rows: one MMA with M = 128 (dj = 0, 1) and one with M = 64 (dj = 2, A two positions further)
  constexpr uint32_t PX = 2u * CIN, PY = 2u * COUT;
  constexpr uint32_t SWX = CIN == 16 ? 6u : (CIN == 32 ? 4u : 2u), SWY = COUT == 16 ? 6u : (COUT == 32 ? 4u : 2u);
  constexpr uint32_t NACCC = (TWO ? 6u : 3u) * COUT, TCOLS = NACCC <= 128 ? 128u : (NACCC <= 256 ? 256u : 512u);
  constexpr int YC8 = COUT / 8;
  __shared__ __align__(8) uint64_t bars[3 * SW_MAX_STAGES + 1];      // raw[3], full[3], sempty[3], done
  __shared__ uint32_t tmem_base_smem;
  const int tid = threadIdx.x, warp = tid >> 5, NS = a.nstages;
  uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  const int Wp = a.W + 2, Rb = (a.R + 2) * Wp;
  const uint32_t bar0 = smem_u32(&bars[0]);
  auto RAW = [&](int s) { return bar0 + 8u * (uint32_t)s; };
  auto FULL = [&](int s) { return bar0 + 8u * (uint32_t)(SW_MAX_STAGES + s); };
  auto SEMPTY = [&](int s) { return bar0 + 8u * (uint32_t)(2 * SW_MAX_STAGES + s); };
  const uint32_t DONE = bar0 + 8u * (3 * SW_MAX_STAGES);
  if (tid == 0) {
    for (int i = 0; i < 3 * SW_MAX_STAGES + 1; ++i)
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" :: "r"(bar0 + 8u * i), "r"((i >= 2 * SW_MAX_STAGES && i < 3 * SW_MAX_STAGES) ? 2 : 1) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    tma::prefetch_map(&xmap); tma::prefetch_map(&ymap);
  }
  if (warp == NLOAD / 32) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" :: "r"(smem_u32(&tmem_base_smem)), "r"(TCOLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
  }
  // everything outside the landed boxes (slack positions, DY rows below a band) stays zero for the whole kernel
  for (uint32_t i = tid; i < a.stage_bytes * (uint32_t)NS / 16; i += NLOAD + 64) reinterpret_cast<uint4*>(smem)[i] = make_uint4(0, 0, 0, 0);
  asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
  const uint32_t tmem_base = tmem_base_smem;
  const int ngroups = (a.F + a.G - 1) / a.G, nitems = ngroups * a.nbands;
  const int my_items = ((int)blockIdx.x < nitems) ? (nitems - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
  float* out = a.partial + (size_t)blockIdx.x * 9 * (CIN + 1) * COUT;

  if (warp < NLOAD / 32) {
    // ================= loaders: ReLU fix-up and bias sums =================
    float db[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) db[k] = 0.f;
    const int c8 = tid % YC8, p0 = tid / YC8, pstep = NLOAD / YC8, ny = a.G * a.dy_rows * Wp;
    for (int it = 0; it < my_items; ++it) {
      const int s = it % NS, use = it / NS;
      if (!mbar_wait(RAW(s), (uint32_t)(use & 1))) { if (a.error_flag) *a.error_flag = 7; }
      uint8_t* xs = smem + (size_t)s * a.stage_bytes; const uint8_t* ys = xs + a.y_off + (size_t)a.dy_off * PY;
      if (a.relu_in) {
        const __nv_bfloat162 z = __float2bfloat162_rn(0.f);
        const int n16 = a.G * Rb * (CIN / 8);
        for (int i = tid; i < n16; i += NLOAD) {      // elementwise: the swizzle does not matter
          uint4* px = reinterpret_cast<uint4*>(xs + (size_t)a.x_off * PX) + i;
          uint4 v = *px;
          __nv_bfloat162* h = reinterpret_cast<__nv_bfloat162*>(&v);
#pragma unroll
          for (int k = 0; k < 4; ++k) h[k] = __hmax2(h[k], z);
          *px = v;
        }
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
        asm volatile("bar.sync 1, %0;\n" :: "n"(NLOAD) : "memory");
        if (tid == 0) mbar_arrive(FULL(s));
      }
      const uint32_t ybase = smem_u32(ys);
      for (int p = p0; p < ny; p += pstep) {          // logical chunk c8 of row p sits at physical chunk c8 ^ (address bits 7..)
        const uint32_t row = ybase + (uint32_t)p * PY, phys = (uint32_t)c8 ^ ((row >> 7) & (uint32_t)(YC8 - 1));
        const uint4 v = *reinterpret_cast<const uint4*>(ys + (size_t)p * PY + phys * 16);
        const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&v);
#pragma unroll
        for (int k = 0; k < 4; ++k) { const float2 f = __bfloat1622float2(h[k]); db[2 * k] += f.x; db[2 * k + 1] += f.y; }
      }
      asm volatile("bar.sync 1, %0;\n" :: "n"(NLOAD) : "memory");
      if (tid == 0) mbar_arrive(SEMPTY(s));
    }
    // ---- all MMAs complete: accumulators final, shared memory free ----
    if (my_items > 0 && !mbar_wait(DONE, 0u)) { if (a.error_flag) *a.error_flag = 2; }
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
    float* dbs = reinterpret_cast<float*>(smem);      // [NLOAD][8]
#pragma unroll
    for (int k = 0; k < 8; ++k) dbs[tid * 8 + k] = db[k];
    asm volatile("bar.sync 1, %0;\n" :: "n"(NLOAD) : "memory");
    if (tid < COUT) {      // threads with chunk tid/8, in thread order: a fixed association
      float t = 0.f;
      for (int j = 0; j < pstep; ++j) t += dbs[(j * YC8 + tid / 8) * 8 + (tid % 8)];
      out[(size_t)CIN * COUT + tid] = t;              // tap 0, row CIN = the bias gradient
    }
    if (warp < 4) {
      const int lane = tid & 31;
      // accumulator rows: M = 128 -> row = TMEM lane; M = 64 -> row r sits in lane 32*(r/16) + r%16
      const int row128 = tid, row64 = (lane < 16) ? warp * 16 + lane : 1 << 20;
      for (int part = 0; part < (TWO ? 2 : 1); ++part) {
        const int um = (TWO && part == 1) ? 64 : UM;
        const int row = um == 128 ? row128 : row64;
        const int nrows = TWO ? (part == 0 ? 128 : 64) : 3 * CIN, dj0 = part * 2;
        const bool warp_needed = um == 128 ? (warp * 32 < nrows) : (warp * 16 < nrows);
        if (!warp_needed) continue;
        for (int acc = 0; acc < 3; ++acc) {
#pragma unroll
          for (int c0 = 0; c0 < COUT; c0 += 16) {
            float v[16];
            tmem_ld16(tmem_base + ((uint32_t)(warp * 32) << 16) + (uint32_t)(part * 3 * COUT + acc * COUT + c0), v);
            if (row >= nrows) continue;
            const int tap = (2 - acc) * 3 + dj0 + row / CIN, r = row % CIN;      // column group e = acc holds the tap row di = 2 - e
#pragma unroll
            for (int i = 0; i < 16; ++i) out[((size_t)tap * (CIN + 1) + r) * COUT + c0 + i] = v[i];
          }
        }
      }
    }
  } else if (warp == NLOAD / 32) {
    // ================= MMA issuer =================
    const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | (1u << 15) | (1u << 16) | ((uint32_t)((3 * COUT) >> 3) << 17) | ((uint32_t)(UM >> 4) << 24);
    const uint32_t idesc64 = (idesc & ~(0x1Fu << 24)) | ((uint32_t)(64 >> 4) << 24);
    const uint32_t a_hi = ((8u * PX) >> 4) | (1u << 14) | (SWX << 29), b_hi = ((8u * PY) >> 4) | (1u << 14) | (SWY << 29);
    // K runs over stored DY rows r: column group e reads row r + e*Wp = DY position r + e*Wp - dy_off, A reads X position
    // r - (dy_off - 2*Wp) + dj; with p = r + e*Wp - dy_off this is X[p + (2-e)*Wp + dj] * DY[p]: tap (2-e, dj)
    const int r_begin = ((a.dy_off - 2 * Wp) / 16) * 16, r_end = a.kext + a.dy_off;
    uint32_t accumulate = 0;
    for (int it = 0; it < my_items; ++it) {
      const int s = it % NS, use = it / NS;
      if (!mbar_wait(a.relu_in ? FULL(s) : RAW(s), (uint32_t)(use & 1))) { if (a.error_flag) *a.error_flag = 2; }
      asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
      const uint32_t x_base = smem_u32(smem) + (uint32_t)s * a.stage_bytes, y_base = x_base + a.y_off;
      uint32_t xl = (((x_base >> 4) & 0x3FFFu) | ((PX >> 4) << 16)) + (uint32_t)(a.x_off + r_begin - (a.dy_off - 2 * Wp)) * (PX >> 4);      // LBO = one position
      uint32_t yl = (((y_base >> 4) & 0x3FFFu) | ((((uint32_t)Wp * PY) >> 4) << 16)) + (uint32_t)r_begin * (PY >> 4);           // LBO = one image row
#pragma unroll 4
      for (int r = r_begin; r < r_end; r += 16) {
        if (elect_one()) mma_f16(tmem_base, ((uint64_t)a_hi << 32) | xl, ((uint64_t)b_hi << 32) | yl, idesc, accumulate);
        if (TWO) { if (elect_one()) mma_f16(tmem_base + 3u * COUT, ((uint64_t)a_hi << 32) | (xl + 2u * (PX >> 4)), ((uint64_t)b_hi << 32) | yl, idesc64, accumulate); }
        accumulate = 1;
        xl += PX; yl += PY;      // 16 positions * (pitch / 16)
      }
      if (elect_one()) mma_commit(SEMPTY(s));
      __syncwarp();
    }
    if (elect_one()) mma_commit(DONE);
    __syncwarp();
  } else if (tid == NLOAD + 32) {
    // ================= TMA producer =================
    const uint32_t xbytes = (uint32_t)(a.G * Rb) * PX, ybytes = (uint32_t)(a.G * a.dy_rows * Wp) * PY;
    for (int it = 0; it < my_items; ++it) {
      const int item = blockIdx.x + it * gridDim.x, s = it % NS, use = it / NS;
      if (use > 0 && !mbar_wait(SEMPTY(s), (uint32_t)((use - 1) & 1))) { if (a.error_flag) *a.error_flag = 7; }
      const int grp = item / a.nbands, band = item - grp * a.nbands, f0 = grp * a.G, yb = band * a.R;
      const uint32_t xs = smem_u32(smem) + (uint32_t)s * a.stage_bytes;
      tma::arrive_expect_tx(RAW(s), xbytes + ybytes);
      tma::load_4d(xs + (uint32_t)a.x_off * PX, &xmap, 0, -1, yb - 1, f0, RAW(s));
      tma::load_4d(xs + a.y_off + (uint32_t)a.dy_off * PY, &ymap, 0, 0, yb, f0, RAW(s));
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  if (warp == NLOAD / 32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" :: "r"(tmem_base), "r"(TCOLS) : "memory");
}

}  // namespace tcw

bool wgrad_tc_supported(const Geom& g) {
  // Cin = 64 runs as two launches over 32 input channels each; Cin = 16 supports Cout <= 32
  const bool okc = (g.Cin == 16 && (g.Cout == 16 || g.Cout == 32)) || ((g.Cin == 32 || g.Cin == 64) && (g.Cout == 16 || g.Cout == 32 || g.Cout == 64));
  return g.kh == 3 && g.kw == 3 && g.s == 1 && g.p == 1 && okc && g.H == g.Ho && g.W == g.Wo;
}

constexpr int WGRAD_TC_MAX_CTAS = 148;
size_t wgrad_tc_partial_elems(const Geom& g) { return (size_t)WGRAD_TC_MAX_CTAS * 9 * (g.Cin + 1) * g.Cout; }

// 3-tap stacking needs 3*Cin+1 accumulator rows: UMMA M = 64 for Cin = 16, M = 128 for Cin = 32
constexpr int wgrad_um(int cin) { return cin == 16 ? 64 : 128; }

struct WPlan { int G, R, nbands, npix_alloc, kext, stage_planes; size_t smem; };
static WPlan wgrad_plan(int H, int W, int cin, int cout) {
  const int xpl = 3 * (cin / 8), WGRAD_UM = wgrad_um(cin);
  const int Wp = W + 2, slack = 2 * Wp + 2;
  WPlan p;
  p.stage_planes = std::max(WGRAD_UM / 8, xpl + 1 + cout / 8);
  const int total_planes = p.stage_planes + std::max(p.stage_planes, WGRAD_UM / 8);
  const int maxpix = (216 * 1024) / (16 * total_planes);
  if ((H + 2) * Wp + slack + 16 <= maxpix) {
    p.R = H; p.nbands = 1; p.G = std::min(8, (maxpix - slack - 16) / ((H + 2) * Wp));
  } else {
    int rmax = (maxpix - slack - 16) / Wp - 2; if (rmax < 1) rmax = 1;
    p.G = 1; p.nbands = (H + rmax - 1) / rmax; p.R = (H + p.nbands - 1) / p.nbands;
  }
  p.kext = (p.G * (p.R + 2) * Wp + 15) / 16 * 16;
  p.npix_alloc = (p.kext + slack + 7) / 8 * 8;
  p.smem = (size_t)total_planes * p.npix_alloc * 16;
  return p;
}

template <int CIN, int COUT>
static int launch_w(const tcw::WgradTcArgs& a, const CUtensorMap& xmap, const CUtensorMap& ymap, size_t smem, int grid, cudaStream_t st) {
  { int rc = ensure_dyn_smem((const void*)tcw::wgrad3x3_tc_kernel<CIN, COUT, wgrad_um(CIN), true>, smem); if (rc) return rc; }
  tcw::wgrad3x3_tc_kernel<CIN, COUT, wgrad_um(CIN), true><<<grid, tcw::NLOAD + 64, smem, st>>>(a, xmap, ymap);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

// plan of the swizzled kernel: 2 stages of G whole frames (or one row band) in <= 208 KB (measured: two large stages beat three or
// four smaller ones, the per-item hand-off costs more than the extra depth buys); a function of the shape only
struct SwPlan { int G, R, nbands, npix_alloc, kext, nstages; size_t stage_bytes, y_off, smem; bool ok; int dy_off, x_off; };
static SwPlan sw_plan(int F, int H, int W, int cin, int cout) {
  const int Wp = W + 2;
  const size_t avail = (size_t)208 * 1024 / 2;
  auto a1k = [](size_t b) { return (b + 1023) & ~(size_t)1023; };
  const int px = 2 * cin, py = 2 * cout;
  const int x_off = std::max(16, 1024 / px), per = 1024 / py, dy_off = (2 * Wp + per - 1) / per * per;      // both keep the landed boxes 1024-byte aligned
  auto stage = [&](int npos, int* kext, int* npix) {
    *kext = (npos + 15) / 16 * 16; *npix = *kext + 2 * Wp + 8;
    return a1k((size_t)(x_off + *npix) * px) + a1k((size_t)(dy_off + *npix) * py);
  };
  SwPlan p{1, H, 1, 0, 0, 2, 0, 0, 0, true};
  int kx, np;
  if (stage((H + 2) * Wp, &kx, &np) <= avail) {
    long best = -1;
    for (int G = 1; G <= 8 && stage(G * (H + 2) * Wp, &kx, &np) <= avail; ++G) {
      const long items = (F + G - 1) / G, per_cta = (items + 147) / 148, cost = per_cta * ((long)G * (H + 2) * Wp + 600);
      if (best < 0 || cost < best) { best = cost; p.G = G; }
    }
  } else {
    int rows = H;
    while (rows > 1 && stage((rows + 2) * Wp, &kx, &np) > avail) --rows;
    if (stage((rows + 2) * Wp, &kx, &np) > avail) { p.ok = false; return p; }
    p.nbands = (H + rows - 1) / rows; p.R = (H + p.nbands - 1) / p.nbands;
  }
  p.stage_bytes = stage(p.G * (p.R + 2) * Wp, &p.kext, &p.npix_alloc);
  p.y_off = a1k((size_t)(x_off + p.npix_alloc) * px);
  p.dy_off = dy_off; p.x_off = x_off;
  p.smem = 1024 + (size_t)p.nstages * p.stage_bytes;
  return p;
}

template <int CIN, int COUT>
static int launch_sw(const tcw::WgradSwArgs& a, const CUtensorMap& xmap, const CUtensorMap& ymap, size_t smem, int grid, cudaStream_t st) {
  { int rc = ensure_dyn_smem((const void*)tcw::wgrad3x3_sw_kernel<CIN, COUT>, smem); if (rc) return rc; }
  tcw::wgrad3x3_sw_kernel<CIN, COUT><<<grid, tcw::NLOAD + 64, smem, st>>>(a, xmap, ymap);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

int launch_wgrad_reduce_batch(const WgradReduceBatch& b, float* grad, cudaStream_t st) {
  if (b.n == 0) return CB_OK;
  tcw::wgrad_tc_reduce_batch_kernel<<<b.blocks, tcw::RL * tcw::RB, 0, st>>>(b, grad);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

int launch_wgrad_tc(const Geom& g, const ParamMap& pm, int F, const bf16* x, const bf16* dy, bool relu_in, float* partial, float* grad,
                    int* error_flag, cudaStream_t st, WgradReduceBatch* defer) {
  if (F <= 0) return CB_OK;
  if (g.Cin == 16 || g.Cin == 32 || g.Cin == 64) {      // swizzled whole-pixel staging
    const SwPlan q = sw_plan(F, g.H, g.W, g.Cin, g.Cout);
    const int dy_rows = q.nbands > 1 ? q.R : q.R + 2;
    CUtensorMap xmap, ymap; memset(&xmap, 0, sizeof xmap); memset(&ymap, 0, sizeof ymap);
    if (q.ok && g.W + 2 <= 256 && q.R + 2 <= 256 && tma::make_nhwc_map(&xmap, x, F, g.H, g.W, g.Cin, g.W + 2, q.R + 2, q.G, g.Cin, true) &&
        tma::make_nhwc_map(&ymap, dy, F, g.H, g.W, g.Cout, g.W + 2, dy_rows, q.G, g.Cout, true)) {
      const int nitems = ((F + q.G - 1) / q.G) * q.nbands, grid = std::min(nitems, WGRAD_TC_MAX_CTAS);
      tcw::WgradSwArgs a{partial, F, g.H, g.W, q.G, q.R, q.nbands, q.npix_alloc, q.kext, relu_in ? 1 : 0, dy_rows, q.nstages,
                         (uint32_t)q.stage_bytes, (uint32_t)q.y_off, q.dy_off, q.x_off, error_flag};
      int rc;
      if (g.Cin == 16 && g.Cout == 16) rc = launch_sw<16, 16>(a, xmap, ymap, q.smem, grid, st);
      else if (g.Cin == 16) rc = launch_sw<16, 32>(a, xmap, ymap, q.smem, grid, st);
      else if (g.Cin == 32 && g.Cout == 16) rc = launch_sw<32, 16>(a, xmap, ymap, q.smem, grid, st);
      else if (g.Cin == 32 && g.Cout == 32) rc = launch_sw<32, 32>(a, xmap, ymap, q.smem, grid, st);
      else if (g.Cin == 32) rc = launch_sw<32, 64>(a, xmap, ymap, q.smem, grid, st);
      else if (g.Cout == 16) rc = launch_sw<64, 16>(a, xmap, ymap, q.smem, grid, st);
      else if (g.Cout == 32) rc = launch_sw<64, 32>(a, xmap, ymap, q.smem, grid, st);
      else rc = launch_sw<64, 64>(a, xmap, ymap, q.smem, grid, st);
      if (rc) return rc;
      if (defer && defer->n < WGRAD_MAX_JOBS) {
        defer->job[defer->n++] = WgradReduceJob{partial, grid, g.Cin, 0, defer->blocks, g, pm};
        defer->blocks += (9 * (g.Cin + 1) * g.Cout + tcw::RB - 1) / tcw::RB;
        return CB_OK;
      }
      tcw::wgrad_tc_reduce_kernel<<<(tcw::RL * 9 * (g.Cin + 1) * g.Cout + 255) / 256, 256, 0, st>>>(partial, grid, g, pm, g.Cin, 0, grad);
      CB_CUDA(cudaGetLastError());
      return CB_OK;
    }
  }
  const int cin_k = g.Cin == 64 ? 32 : g.Cin;      // channels per kernel launch
  WPlan p = wgrad_plan(g.H, g.W, cin_k, g.Cout);
  if (p.smem > 224 * 1024) { set_error("wgrad_tc: plan does not fit shared memory"); return CB_EINVAL; }
  const int nitems = ((F + p.G - 1) / p.G) * p.nbands;
  const int grid = std::min(nitems, WGRAD_TC_MAX_CTAS);
  // TMA boxes: X [8][W+2][R+2][G] started at (-1+dj, yb-1); DY [8][W+2][rows][G] started at (0, yb) with rows = R for banded
  // plans (G = 1: the rows below the band must stay zero) and R+2 = H+2 for whole frames (out-of-bounds rows are zero-filled)
  const int dy_rows = p.nbands > 1 ? p.R : p.R + 2;
  CUtensorMap xmap, ymap; memset(&xmap, 0, sizeof xmap); memset(&ymap, 0, sizeof ymap);
  const bool use_tma = g.W + 2 <= 256 && p.R + 2 <= 256 && tma::make_nhwc_map(&xmap, x, F, g.H, g.W, g.Cin, g.W + 2, p.R + 2, p.G) &&
                       tma::make_nhwc_map(&ymap, dy, F, g.H, g.W, g.Cout, g.W + 2, dy_rows, p.G);
  for (int c_off = 0; c_off < g.Cin; c_off += cin_k) {
    tcw::WgradTcArgs a{x, dy, partial, F, g.H, g.W, p.G, p.R, p.nbands, p.npix_alloc, p.kext, relu_in ? 1 : 0, p.stage_planes, use_tma ? 1 : 0, dy_rows,
                       use_tma ? 1 : 0, c_off, g.Cin, error_flag};
    int rc;
    if (cin_k == 16 && g.Cout == 16) rc = launch_w<16, 16>(a, xmap, ymap, p.smem, grid, st);
    else if (cin_k == 16) rc = launch_w<16, 32>(a, xmap, ymap, p.smem, grid, st);
    else if (g.Cout == 16) rc = launch_w<32, 16>(a, xmap, ymap, p.smem, grid, st);
    else if (g.Cout == 32) rc = launch_w<32, 32>(a, xmap, ymap, p.smem, grid, st);
    else rc = launch_w<32, 64>(a, xmap, ymap, p.smem, grid, st);
    if (rc) return rc;
    tcw::wgrad_tc_reduce_kernel<<<(tcw::RL * 9 * (cin_k + 1) * g.Cout + 255) / 256, 256, 0, st>>>(partial, grid, g, pm, cin_k, c_off, grad);
    CB_CUDA(cudaGetLastError());
  }
  return CB_OK;
}

}  // namespace cb
