// Stage convolution of the IMPALA-ResNet fused with the max-pool that follows it (conv3x3 pad 1 -> max-pool 3x3 s2 SAME),
// CB_PREC_BF16_TC, forward only.  The conv output of a stage is consumed by nothing but its pool (the pool's adjoint needs only the stored
// arg-max), so it never has to reach HBM: a persistent warp-specialised CTA per SM computes a band of 2 Rp + 1 conv rows with tcgen05 into
// TMEM, drains it (+ bias, bf16) into a swizzled shared-memory band and pools Rp rows out of it.  Same item pipeline as the first layer's
// kernel (conv0_tc.cu), same operand scheme as conv3x3_tc_pipe_kernel (conv_tc.cu):
//   warp  0      TMA producer: one 4-D box [Cin][W+2][R+2][1] started at (-1, yb-1) lands a band with its zero halo, whole pixels in swizzled rows
//   warp  1      MMA issuer:   9 Cin/16 tcgen05.mma per 128-position tile (a tap = a constant shift of the A descriptor's start address)
//   warps 2-9    epilogue:     TMEM -> + bias -> bf16 conv band ctile[s]
//   warps 10-21  pool:         3x3 s2 SAME max + first arg-max (A10, A11) -> pooled map, arg-max bytes
// mbarriers (two items deep): LFULL[s] (TMA bytes) <- LEMPTY[s] (MMA commit); TFULL[s] (commit) <- TEMPTY[s] (8 arrivals);
//                             CFULL[s] (8 arrivals) <- CEMPTY[s] (12 arrivals).
#include "common.cuh"
#include "tma.cuh"
#include "tc_ptx.cuh"
#include "pool.cuh"

#include <cstring>

namespace cb {
namespace tcp {
using namespace ptx;

constexpr int EPI_WARPS = 8, POOL_WARPS = 12, THREADS = (2 + EPI_WARPS + POOL_WARPS) * 32;
struct Args {
  const bf16* w; const float* bias; bf16* pool_out; uint8_t* pool_arg;
  int F, H, W, R, Rp, nbands; uint32_t stage_bytes, ctile_bytes; int* error_flag;
};
__device__ __forceinline__ void arrive(uint32_t bar) { asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}\n" :: "r"(bar) : "memory"); }

template <int CIN, int COUT>
__global__ void __launch_bounds__(THREADS, 1) conv3x3_pool_kernel(const Args a, const __grid_constant__ CUtensorMap tmap) {
  extern __shared__ __align__(128) uint8_t smem[];
  constexpr int NCH = CIN / 8, KSTEPS = CIN / 16;
  constexpr uint32_t W_BYTES = 9u * CIN * COUT * 2u, PITCH = 2u * CIN, SWZ = CIN == 16 ? 6u : (CIN == 32 ? 4u : 2u);
  __shared__ __align__(8) uint64_t bars[12];
  __shared__ uint32_t tmem_base_smem;
  __shared__ __align__(16) float bias_s[64];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, Wp = a.W + 2;
  const uint32_t bar0 = smem_u32(&bars[0]);
  auto LFULL = [&](int s) { return bar0 + 8u * (uint32_t)s; };        auto LEMPTY = [&](int s) { return bar0 + 8u * (uint32_t)(2 + s); };
  auto TFULL = [&](int s) { return bar0 + 8u * (uint32_t)(4 + s); };  auto TEMPTY = [&](int s) { return bar0 + 8u * (uint32_t)(6 + s); };
  auto CFULL = [&](int s) { return bar0 + 8u * (uint32_t)(8 + s); };  auto CEMPTY = [&](int s) { return bar0 + 8u * (uint32_t)(10 + s); };
  uint8_t* w_smem = smem;
  uint8_t* stages = smem + W_BYTES; stages += (1024u - (smem_u32(stages) & 1023u)) & 1023u;      // the swizzle is a function of the absolute address
  uint8_t* ctiles = stages + 2 * (size_t)a.stage_bytes;
  if (tid == 0) {
    for (int s = 0; s < 2; ++s) {
      mbar_init(LFULL(s), 1); mbar_init(LEMPTY(s), 1); mbar_init(TFULL(s), 1); mbar_init(TEMPTY(s), EPI_WARPS);
      mbar_init(CFULL(s), EPI_WARPS); mbar_init(CEMPTY(s), POOL_WARPS);
    }
    tma::prefetch_map(&tmap);
  }
  if (warp == 1) tmem_alloc(smem_u32(&tmem_base_smem), 512);
  for (uint32_t i = tid; i < 2 * a.stage_bytes / 16; i += THREADS) reinterpret_cast<uint4*>(stages)[i] = make_uint4(0, 0, 0, 0);      // slack rows beyond the box stay zero
  pdl_wait(); pdl_trigger();
  if (tid < COUT) bias_s[tid] = a.bias[tid];
  for (uint32_t i = tid; i < W_BYTES / 16; i += THREADS) reinterpret_cast<uint4*>(w_smem)[i] = reinterpret_cast<const uint4*>(a.w)[i];
  fence_async_smem();
  tc_fence_before(); __syncthreads(); tc_fence_after();
  const uint32_t tmem_base = tmem_base_smem;
  const int nitems = a.F * a.nbands;
  const int my_items = ((int)blockIdx.x < nitems) ? (nitems - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
  const int Ho = (a.H + 1) / 2, Wo = (a.W + 1) / 2;
  int th_ = (Ho - 1) * 2 + 3 - a.H; if (th_ < 0) th_ = 0; const int ph = th_ / 2;
  int tw_ = (Wo - 1) * 2 + 3 - a.W; if (tw_ < 0) tw_ = 0; const int pw = tw_ / 2;
  const int ntiles = (a.R * Wp + 127) / 128;
  auto item_geom = [&](int it, int& f, int& py0, int& yb) {
    const int item = blockIdx.x + it * gridDim.x; f = item / a.nbands; const int band = item - f * a.nbands;
    py0 = band * a.Rp; yb = max(0, 2 * py0 - ph);
  };

  if (warp == 0) {
    // ================= TMA producer =================
    const uint32_t bytes = (uint32_t)((a.R + 2) * Wp) * PITCH;
    for (int it = 0; it < my_items; ++it) {
      const int s = it & 1, use = it >> 1; int f, py0, yb; item_geom(it, f, py0, yb);
      if (use > 0 && !mbar_wait(LEMPTY(s), (uint32_t)((use - 1) & 1))) { if (a.error_flag) *a.error_flag = 8; }
      if (elect_one()) {
        tma::arrive_expect_tx(LFULL(s), bytes);
        tma::load_4d(smem_u32(stages) + (uint32_t)s * a.stage_bytes, &tmap, 0, -1, yb - 1, f, LFULL(s));
      }
      __syncwarp();
    }
  } else if (warp == 1) {
    // ================= MMA issuer =================
    const uint32_t idesc = make_idesc(128, COUT, 0, 0);
    const uint32_t d_hi = 8u | (1u << 14);                                                      // B: SBO = 128 B
    const uint32_t a_hi = ((8u * PITCH) >> 4) | (1u << 14) | (SWZ << 29);                       // A: SBO = 8 rows, swizzle mode in bits 61-63
    const uint32_t b_lo = ((smem_u32(w_smem) >> 4) & 0x3FFFu) | ((uint32_t)COUT << 16);         // LBO = COUT*16 B
    for (int it = 0; it < my_items; ++it) {
      const int s = it & 1, use = it >> 1;
      if (!mbar_wait(LFULL(s), (uint32_t)(use & 1))) { if (a.error_flag) *a.error_flag = 8; }
      if (use > 0 && !mbar_wait(TEMPTY(s), (uint32_t)((use - 1) & 1))) { if (a.error_flag) *a.error_flag = 8; }
      tc_fence_after();
      const uint32_t a_lo = (((smem_u32(stages) + (uint32_t)s * a.stage_bytes) >> 4) & 0x3FFFu) | (1u << 16);
#pragma unroll 1
      for (int t = 0; t < ntiles; ++t) {
        const uint32_t td = tmem_base + (uint32_t)(s * 256 + t * COUT);
        uint32_t row_lo = a_lo + (uint32_t)t * 128u * (PITCH >> 4);
#pragma unroll
        for (int di = 0; di < 3; ++di) {
#pragma unroll
          for (int dj = 0; dj < 3; ++dj) {
#pragma unroll
            for (int ks = 0; ks < KSTEPS; ++ks) {
              const uint64_t ad = ((uint64_t)a_hi << 32) | (uint64_t)(row_lo + (uint32_t)(dj * (PITCH >> 4) + 2 * ks));
              const uint64_t bd = ((uint64_t)d_hi << 32) | (uint64_t)(b_lo + (uint32_t)(((di * 3 + dj) * NCH + 2 * ks) * COUT));
              if (elect_one()) mma_f16(td, ad, bd, idesc, (di | dj | ks) ? 1u : 0u);
            }
          }
          row_lo += (uint32_t)Wp * (PITCH >> 4);
        }
      }
      if (elect_one()) { mma_commit(TFULL(s)); mma_commit(LEMPTY(s)); }
      __syncwarp();
    }
  } else if (warp < 2 + EPI_WARPS) {
    // ================= epilogue: warp e drains lanes 32 (warp % 4) .. +31 of every second tile =================
    const int e = warp - 2, q4 = warp & 3, half = e >> 2;
    const uint32_t magic_Wp = (uint32_t)((0x100000000ull + (uint64_t)Wp - 1) / (uint64_t)Wp);
    for (int it = 0; it < my_items; ++it) {
      const int s = it & 1, use = it >> 1; int f, py0, yb; item_geom(it, f, py0, yb);
      if (!mbar_wait(TFULL(s), (uint32_t)(use & 1))) { if (a.error_flag) *a.error_flag = 8; }
      if (use > 0 && !mbar_wait(CEMPTY(s), (uint32_t)((use - 1) & 1))) { if (a.error_flag) *a.error_flag = 8; }
      tc_fence_after();
      uint8_t* ct = ctiles + (size_t)s * a.ctile_bytes;
      for (int t = half; t < ntiles; t += 2) {
        const int q = t * 128 + q4 * 32 + lane, yl = (int)__umulhi((uint32_t)q, magic_Wp), x = q - yl * Wp, y = yb + yl;
        const bool valid = yl < a.R && y < a.H && x < a.W;
#pragma unroll
        for (int c0 = 0; c0 < COUT; c0 += 16) {
          float v[16];
          tmem_ld16(tmem_base + ((uint32_t)(q4 * 32) << 16) + (uint32_t)(s * 256 + t * COUT + c0), v);
          if (!valid) continue;
          uint4 o0, o1;
          __nv_bfloat162* p0 = reinterpret_cast<__nv_bfloat162*>(&o0); __nv_bfloat162* p1 = reinterpret_cast<__nv_bfloat162*>(&o1);
#pragma unroll
          for (int i = 0; i < 16; i += 4) { const float4 b4 = *reinterpret_cast<const float4*>(bias_s + c0 + i); v[i] += b4.x; v[i + 1] += b4.y; v[i + 2] += b4.z; v[i + 3] += b4.w; }
#pragma unroll
          for (int i = 0; i < 4; ++i) { p0[i] = __floats2bfloat162_rn(v[2 * i], v[2 * i + 1]); p1[i] = __floats2bfloat162_rn(v[8 + 2 * i], v[8 + 2 * i + 1]); }
          const uint32_t off = (uint32_t)(((yl * a.W + x) * COUT + c0) * 2);
          *reinterpret_cast<uint4*>(ct + pool::ct_swz<COUT>(off)) = o0;
          *reinterpret_cast<uint4*>(ct + pool::ct_swz<COUT>(off + 16)) = o1;
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) { arrive(TEMPTY(s)); arrive(CFULL(s)); }
    }
  } else {
    // ================= pool =================
    const int pt = tid - (2 + EPI_WARPS) * 32;
    for (int it = 0; it < my_items; ++it) {
      const int s = it & 1, use = it >> 1; int f, py0, yb; item_geom(it, f, py0, yb);
      if (!mbar_wait(CFULL(s), (uint32_t)(use & 1))) { if (a.error_flag) *a.error_flag = 8; }
      pool::pool_band<COUT>(ctiles + (size_t)s * a.ctile_bytes, yb, py0, min(a.Rp, Ho - py0), f, a.H, a.W, Ho, Wo, ph, pw, a.pool_out, a.pool_arg, pt, POOL_WARPS * 32);
      __syncwarp();
      if (lane == 0) arrive(CEMPTY(s));
    }
  }
  tc_fence_before(); __syncthreads();
  if (warp == 1) tmem_dealloc(tmem_base, 512);
}

}  // namespace tcp

// plan: the largest band of Rp pooled rows whose tiles fit one 256-column TMEM buffer and whose two stages + two conv bands + weights fit 200 KB
struct ConvPoolPlan { int Rp, R, nbands; size_t stage_bytes, ctile_bytes, smem; bool ok; };
static ConvPoolPlan conv_pool_plan(int H, int W, int cin, int cout) {
  const int Wp = W + 2, Ho = (H + 1) / 2;
  const size_t wbytes = (size_t)9 * cin * cout * 2;
  auto tiles_of = [&](int rp) { return ((2 * rp + 1) * Wp + 127) / 128; };
  auto stage_of = [&](int rp) { return ((size_t)(tiles_of(rp) * 128 + 2 * Wp + 8) * cin * 2 + 1023) & ~(size_t)1023; };
  auto ctile_of = [&](int rp) { return ((size_t)(2 * rp + 1) * W * cout * 2 + 127) & ~(size_t)127; };
  auto smem_of = [&](int rp) { return wbytes + 1024 + 2 * stage_of(rp) + 2 * ctile_of(rp); };
  auto fits = [&](int rp) { return tiles_of(rp) * cout <= 256 && smem_of(rp) <= (size_t)200 * 1024 && 2 * rp + 3 <= 256; };
  ConvPoolPlan p{1, 3, Ho, 0, 0, 0, false};
  if (!fits(1)) return p;
  int rp = 1; while (rp < Ho && fits(rp + 1)) ++rp;
  p.nbands = (Ho + rp - 1) / rp; p.Rp = (Ho + p.nbands - 1) / p.nbands; p.R = 2 * p.Rp + 1;
  p.stage_bytes = stage_of(p.Rp); p.ctile_bytes = ctile_of(p.Rp); p.smem = smem_of(p.Rp); p.ok = true;
  return p;
}

bool conv_pool_tc_supported(const Geom& g) {
  auto okc = [](int c) { return c == 16 || c == 32 || c == 64; };
  return g.kh == 3 && g.kw == 3 && g.s == 1 && g.p == 1 && okc(g.Cin) && okc(g.Cout) && g.H == g.Ho && g.W == g.Wo && g.W + 2 <= 256 &&
         tma::encode_fn() != nullptr && conv_pool_plan(g.H, g.W, g.Cin, g.Cout).ok;
}

template <int CIN, int COUT>
static int launch_cp(const tcp::Args& a, const CUtensorMap& tmap, size_t smem, int grid, cudaStream_t st) {
  { int rc = ensure_dyn_smem((const void*)tcp::conv3x3_pool_kernel<CIN, COUT>, smem); if (rc) return rc; }
  CB_CUDA(launch_pdl(tcp::conv3x3_pool_kernel<CIN, COUT>, dim3(grid), dim3(tcp::THREADS), smem, st, a, tmap));
  return CB_OK;
}

// in: [F,H,W,Cin] bf16 (read as stored: the stage conv has no input ReLU); w: the forward B-operand pack of conv_tc.cu; outputs: pooled map
// [F,Ho,Wo,Cout] and arg-max bytes
int launch_conv_pool_tc(const Geom& g, int F, const bf16* in, const bf16* w, const float* bias, bf16* pool_out, uint8_t* pool_arg, int* error_flag, cudaStream_t st) {
  if (F <= 0) return CB_OK;
  const ConvPoolPlan p = conv_pool_plan(g.H, g.W, g.Cin, g.Cout);
  CUtensorMap tmap; memset(&tmap, 0, sizeof tmap);
  if (!p.ok || !tma::make_nhwc_map(&tmap, in, F, g.H, g.W, g.Cin, g.W + 2, p.R + 2, 1, g.Cin, true)) { set_error("conv_pool_tc: no plan, or the driver refused the tensor map"); return CB_ECUDA; }
  tcp::Args a{w, bias, pool_out, pool_arg, F, g.H, g.W, p.R, p.Rp, p.nbands, (uint32_t)p.stage_bytes, (uint32_t)p.ctile_bytes, error_flag};
  const int grid = std::min(F * p.nbands, 148);
#define CB_CP_CASE(ci, co) if (g.Cin == ci && g.Cout == co) return launch_cp<ci, co>(a, tmap, p.smem, grid, st);
  CB_CP_CASE(16, 16) CB_CP_CASE(16, 32) CB_CP_CASE(32, 32) CB_CP_CASE(32, 64) CB_CP_CASE(64, 64) CB_CP_CASE(16, 64) CB_CP_CASE(32, 16) CB_CP_CASE(64, 32) CB_CP_CASE(64, 16)
#undef CB_CP_CASE
  set_error("conv_pool_tc: unsupported channel counts");
  return CB_EINVAL;
}

}  // namespace cb
