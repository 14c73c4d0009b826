// tcgen05 / TMEM weight-gradient kernel for 3x3 stride-1 pad-1 convolutions, CB_PREC_BF16_TC, sm_100a.
//
//   dW[tap][c][o] = sum_q X[q + shift(tap)][c] * DY[q][o]        db[o] = sum_q DY[q][o]
//
// with q running over the pixel-linear positions of conv_tc.cu.  The contraction index is the PIXEL, so both operands are MN-major.
// X and DY are landed once each by TMA as whole pixels (one swizzled shared-memory row per position); the descriptors WALK over that
// single copy (see wgrad3x3_sw_kernel below): ONE tcgen05.mma per 16 positions yields all nine taps.  The accumulator stays in TMEM for
// the whole life of the CTA, which runs over a fixed set of (frame-group, row-band) items and writes ONE fp32 partial [9][Cin+1][Cout]
// at the end; a second kernel adds the partials in CTA order, so the result is bitwise reproducible (no atomics; the item -> CTA map
// depends on the shape only).  Without TMA wgrad_tc_supported() is false and the layer runs on the SIMT split-K GEMM.
#include "common.cuh"
#include "tma.cuh"

#include <cstring>
#include "tc_ptx.cuh"

namespace cb {
namespace tcw {

using namespace ptx;      // tcgen05 / TMEM / mbarrier wrappers: tc_ptx.cuh

constexpr int NLOAD = 256;       // warps 0-7: loaders / bias sums (warps 0-3 later read TMEM); warp 8 issues the MMAs; warp 9 produces
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}\n" :: "r"(bar) : "memory");
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
// The kernel (TMA, Cin in {16, 32, 64}): whole pixels are landed once, one shared-memory row of 2*CIN (X) or 2*COUT (DY)
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
  pdl_wait(); pdl_trigger();      // the prologue above is private to the CTA (tc_ptx.cuh)
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
  return g.kh == 3 && g.kw == 3 && g.s == 1 && g.p == 1 && okc && g.H == g.Ho && g.W == g.Wo && tma::encode_fn() != nullptr;      // TMA-fed only
}

constexpr int WGRAD_TC_MAX_CTAS = 148;
size_t wgrad_tc_partial_elems(const Geom& g) { return (size_t)WGRAD_TC_MAX_CTAS * 9 * (g.Cin + 1) * g.Cout; }

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
  CB_CUDA(launch_pdl(tcw::wgrad3x3_sw_kernel<CIN, COUT>, dim3(grid), dim3(tcw::NLOAD + 64), smem, st, a, xmap, ymap));
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
  set_error("wgrad_tc: no plan for this shape, or the driver refused a tensor map");
  return CB_ECUDA;
}

}  // namespace cb
