// tcgen05 kernels for the FIRST layer of the IMPALA-ResNet in CB_PREC_BF16_TC: 3x3 stride-1 pad-1 conv on
// uint8 NCHW frames with Cin <= 4, forward and weight gradient.  The /255
// normalisation is fused: the raw integers 0..255 (exact in bf16) are the operand and 1/255 scales the
// fp32 accumulator.
//
// Staging: one plane of 16-byte positions [c0 c1 c2 c3 | 1 | 0 0 0] in the pixel-linear order of
// conv_tc.cu (row-band of R rows with its halo).  Channel 4 is the constant 1: its forward weights are
// zero; in the weight gradient it makes row 4 of the accumulator the bias gradient.
//   forward: a K=16 MMA step = two neighbouring positions (taps (di,0),(di,1); then (di,2) + a zero-weight
//            slot): K-major A descriptor with LBO = 16 B, six MMAs per 128-position tile.
//   wgrad:   MN-major A descriptor with SBO = 16 B: the M walk steps over neighbouring positions, so one
//            M = 128 MMA yields the taps (di, 0..2) at rows 8*dj + c; three accumulators [128 x Cout] (one
//            per di) live in TMEM for the life of the CTA; per-CTA partials are summed in CTA order.
#include "common.cuh"
#include "tc_ptx.cuh"
#include "pool.cuh"

namespace cb {
namespace tc0 {
using namespace ptx;

struct Args {
  const uint8_t* obs; const int32_t* frame_idx;   // [*, CIN, H, W] uint8, optional frame gather
  const bf16* w; const float* bias; bf16* out;     // forward: B image [6][2][COUT][8], bias [COUT], out [F,H,W,COUT]
  const bf16* dy; float* partial;                 // wgrad: dy [F,H,W,COUT], partial [grid][3][24][COUT]
  const uint8_t* pool_arg; const bf16* dpool;     // wgrad, fused max-pool adjoint: dy is gathered from dpool [F,Ho,Wo,COUT] through pool_arg
  int F, H, W, CIN, R, nbands, npix_alloc, kext;
  int w_xoff, w_yoff, w_ybytes;   // wgrad: X position p at plane row p + w_xoff; DY position p at row p + w_yoff of the swizzled DY region, w_ybytes per stage
  bf16* pool_out; uint8_t* pool_arg_out; int Rp;  // forward, fused 3x3 s2 SAME max-pool: pooled map + arg-max positions; Rp pooled rows per band
  int* error_flag;
};

// stage rows yb-1 .. yb+R of frame `fr` into the plane (all positions rewritten); the first `npre` quads of this thread may have
// been fetched by the caller (`pre`)
__device__ __forceinline__ void stage_band(const Args& a, uint8_t* xs, size_t fr, int yb, int tid, int nthr = 128, const uint32_t (*pre)[4] = nullptr, int npre = 0) {
  const int Wp = a.W + 2, W4 = a.W / 4, rows = a.R + 2;
  const uint32_t ONE = 0x3F80u;
  int j = 0;
  const uint32_t magic_W4 = (uint32_t)((0x100000000ull + (uint64_t)W4 - 1) / (uint64_t)W4);      // i / W4 = umulhi(i, magic) for i * W4 < 2^32
  for (int i = tid; i < rows * W4; i += nthr, ++j) {
    int lr = (int)__umulhi((uint32_t)i, magic_W4), x0 = (i - lr * W4) * 4, y = yb - 1 + lr;
    uint32_t px[4] = {0, 0, 0, 0};     // per channel: 4 pixels
    if (j == 0 && npre > 0) { px[0] = pre[0][0]; px[1] = pre[0][1]; px[2] = pre[0][2]; px[3] = pre[0][3]; }            // static indices: registers
    else if (j == 1 && npre > 1) { px[0] = pre[1][0]; px[1] = pre[1][1]; px[2] = pre[1][2]; px[3] = pre[1][3]; }
    else if (j == 2 && npre > 2) { px[0] = pre[2][0]; px[1] = pre[2][1]; px[2] = pre[2][2]; px[3] = pre[2][3]; }
    else if ((unsigned)y < (unsigned)a.H)
      for (int c = 0; c < a.CIN; ++c) px[c] = *reinterpret_cast<const uint32_t*>(a.obs + ((fr * a.CIN + c) * a.H + y) * a.W + x0);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      float v0 = (float)((px[0] >> (8 * k)) & 255u), v1 = (float)((px[1] >> (8 * k)) & 255u);
      float v2 = (float)((px[2] >> (8 * k)) & 255u), v3 = (float)((px[3] >> (8 * k)) & 255u);
      __nv_bfloat162 p01 = __floats2bfloat162_rn(v0, v1), p23 = __floats2bfloat162_rn(v2, v3);
      uint4 o; o.x = *reinterpret_cast<uint32_t*>(&p01); o.y = *reinterpret_cast<uint32_t*>(&p23); o.z = ONE; o.w = 0;
      *reinterpret_cast<uint4*>(xs + (size_t)(lr * Wp + x0 + 1 + k) * 16) = o;
    }
  }
  for (int i = tid; i < rows * 2; i += nthr) {       // halo columns
    int lr = i >> 1, xp = (i & 1) ? Wp - 1 : 0;
    *reinterpret_cast<uint4*>(xs + (size_t)(lr * Wp + xp) * 16) = make_uint4(0, 0, ONE, 0);
  }
}

// adjoint of the 3x3 stride-2 SAME max-pool, scatter form, evaluated while staging dy (A11): every pooled
// element adds its gradient to the conv-output pixel its stored arg-max names.  Windows whose (oy, ox)
// parities agree are disjoint (stride 4 between them, width 3), so the four parity classes are applied as
// four barrier-separated phases of plain shared-memory read-modify-writes: no atomics, fixed order,
// bitwise reproducible.  A pixel elected by several windows is rounded to bf16 after each addition.
struct PoolGeom { int Ho, Wo, ph, pw, oy_lo, noy[2], nox[2]; };
__device__ __forceinline__ PoolGeom pool_geom(const Args& a, int yb) {
  PoolGeom q; q.Ho = (a.H + 1) / 2; q.Wo = (a.W + 1) / 2;
  int th = (q.Ho - 1) * 2 + 3 - a.H; if (th < 0) th = 0; q.ph = th / 2;
  int tw = (q.Wo - 1) * 2 + 3 - a.W; if (tw < 0) tw = 0; q.pw = tw / 2;
  int lo = yb + q.ph - 2; lo = lo <= 0 ? 0 : (lo + 1) / 2;
  const int yend = min(yb + a.R, a.H) - 1;
  const int hi = min((yend + q.ph) / 2, q.Ho - 1);
  q.oy_lo = lo;
  for (int par = 0; par < 2; ++par) {
    const int first = lo + (((lo & 1) != par) ? 1 : 0);
    q.noy[par] = hi >= first ? (hi - first) / 2 + 1 : 0;
    q.nox[par] = (q.Wo - par + 1) / 2;
  }
  return q;
}
// item i of phase p -> (oy, ox, ch); returns false past the end
__device__ __forceinline__ bool pool_item(const PoolGeom& q, int p, int i, int ych, int& oy, int& ox, int& ch) {
  const int pa = p >> 1, pb = p & 1, n = q.noy[pa] * q.nox[pb] * ych;
  if (i >= n) return false;
  ch = i % ych; const int r = i / ych; const int ix = r % q.nox[pb], iy = r / q.nox[pb];
  const int first = q.oy_lo + (((q.oy_lo & 1) != pa) ? 1 : 0);
  oy = first + 2 * iy; ox = pb + 2 * ix;
  return true;
}
// DY region of the weight-gradient kernel: one row of PY = 2*COUT bytes per position in the 32B/64B swizzle pattern (16-byte
// chunk c of a row sits at chunk c ^ (address bits 7..)), the layout the MN-major B descriptor with LBO = one image row reads
template <int COUT>
__device__ __forceinline__ uint8_t* dy_chunk(uint8_t* ys, uint32_t ys_addr, int pos, int ch) {
  constexpr uint32_t PY = 2u * COUT;
  const uint32_t row = ys_addr + (uint32_t)pos * PY;
  return ys + (size_t)pos * PY + (((uint32_t)ch ^ ((row >> 7) & (COUT / 8 - 1))) << 4);
}
template <int COUT>
__device__ __forceinline__ void pool_scatter(const Args& a, const PoolGeom& q, uint8_t* ys, uint32_t ys_addr, int yb, int oy, int ox, int ch,
                                             uint2 pk, uint4 dv) {
  const int Wp = a.W + 2, rows = min(a.R, a.H - yb);
  const int y0 = oy * 2 - q.ph - yb, x0 = ox * 2 - q.pw;
  const uint16_t* h = reinterpret_cast<const uint16_t*>(&dv);
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const uint32_t arg = ((k < 4 ? pk.x : pk.y) >> (8 * (k & 3))) & 255u;
    const int wy = (int)((arg * 11u) >> 5), wx = (int)arg - 3 * wy;
    const int yl = y0 + wy;
    if ((unsigned)yl < (unsigned)rows)
      pool::add_bf16(reinterpret_cast<uint16_t*>(dy_chunk<COUT>(ys, ys_addr, yl * Wp + x0 + wx, ch)) + k, h[k]);
  }
}

constexpr int TMEM_COLS = 256;

template <int COUT>
__global__ void __launch_bounds__(256) conv0_fwd_kernel(const Args a) {
  extern __shared__ __align__(128) uint8_t smem[];
  constexpr uint32_t W_BYTES = 6u * 2u * COUT * 16u;
  constexpr int TILES_PER_BATCH = TMEM_COLS / COUT / 2;      // per accumulator half
  __shared__ __align__(8) uint64_t bar_storage[2];
  __shared__ uint32_t tmem_base_smem;
  __shared__ __align__(16) float bias_s[32];
  const int tid = threadIdx.x, warp = tid >> 5, wg = warp >> 2, lane_row = tid & 127, Wp = a.W + 2;      // two warpgroups
  const uint32_t magic_Wp = (uint32_t)((0x100000000ull + (uint64_t)Wp - 1) / (uint64_t)Wp);      // q / Wp = umulhi(q, magic) for q * Wp < 2^32
  if (tid < COUT) bias_s[tid] = a.bias[tid];
  uint8_t* w_smem = smem; uint8_t* xs = smem + W_BYTES;
  const uint32_t bar = smem_u32(&bar_storage[0]);
  if (tid == 0) { mbar_init(bar, 1); mbar_init(bar + 8u, 1); }
  if (warp == 0) tmem_alloc(smem_u32(&tmem_base_smem), TMEM_COLS);
  for (uint32_t i = tid; i < W_BYTES / 16; i += 256) reinterpret_cast<uint4*>(w_smem)[i] = reinterpret_cast<const uint4*>(a.w)[i];
  for (int i = tid; i < a.npix_alloc; i += 256) reinterpret_cast<uint4*>(xs)[i] = make_uint4(0, 0, 0x3F80u, 0);
  tc_fence_before(); __syncthreads(); tc_fence_after();
  const uint32_t tmem_base = tmem_base_smem, idesc = make_idesc(128, COUT, 0, 0);
  const uint32_t a_base = smem_u32(xs), b_base = smem_u32(w_smem);
  uint32_t parity = 0;
  const int nitems = a.F * a.nbands;
  const bool fused = a.pool_out != nullptr;
  const int Ho = (a.H + 1) / 2, Wo = (a.W + 1) / 2;
  int th_ = (Ho - 1) * 2 + 3 - a.H; if (th_ < 0) th_ = 0; const int ph = th_ / 2;
  int tw_ = (Wo - 1) * 2 + 3 - a.W; if (tw_ < 0) tw_ = 0; const int pw = tw_ / 2;
  uint32_t pre[3][4]; int npre = 0;      // this thread's first three observation quads of the NEXT item, fetched while the current one is pooled
  for (int item = blockIdx.x; item < nitems; item += gridDim.x) {
    const int f = item / a.nbands, band = item - f * a.nbands;
    const int py0 = band * a.Rp;                                   // fused: first pooled row of the band
    const int yb = fused ? max(0, 2 * py0 - ph) : band * a.R;      // first conv row computed by this item
    const size_t fr = a.frame_idx ? (size_t)a.frame_idx[f] : (size_t)f;
    stage_band(a, xs, fr, yb, tid, 256, pre, npre);
    fence_async_smem();
    __syncthreads();
    const int ntiles = (a.R * Wp + 127) / 128;
    const int nbatch = (ntiles + TILES_PER_BATCH - 1) / TILES_PER_BATCH;
    // The accumulator is split into two halves of TILES_PER_BATCH tiles: the MMAs of batch k+1 are issued BEFORE batch k is drained, so the
    // tensor core works underneath the epilogue (every operand of the band is already staged).  One mbarrier per half.
    auto issue = [&](int bi) {        // warp 0, converged: one elected lane issues
      const int t0 = bi * TILES_PER_BATCH, nt = min(TILES_PER_BATCH, ntiles - t0), half = bi & 1;
      tc_fence_after();
      const uint32_t a_lo = ((a_base >> 4) & 0x3FFFu) | (1u << 16), a_hi = 8u | (1u << 14);               // LBO 16 B, SBO 128 B
      const uint32_t b_lo = ((b_base >> 4) & 0x3FFFu) | ((uint32_t)COUT << 16), b_hi = 8u | (1u << 14);   // LBO COUT*16 B, SBO 128 B
      for (int s = 0; s < nt; ++s) {
        const uint32_t q0 = (uint32_t)(t0 + s) * 128u;
#pragma unroll
        for (int slot = 0; slot < 6; ++slot) {
          const uint32_t shift = (uint32_t)((slot >> 1) * Wp + (slot & 1) * 2);
          const uint64_t ad = ((uint64_t)a_hi << 32) | (uint64_t)(a_lo + q0 + shift);
          const uint64_t bd = ((uint64_t)b_hi << 32) | (uint64_t)(b_lo + (uint32_t)slot * 2u * COUT);
          if (elect_one()) mma_f16(tmem_base + (uint32_t)((half * TILES_PER_BATCH + s) * COUT), ad, bd, idesc, slot ? 1u : 0u);
        }
      }
      if (elect_one()) mma_commit(bar + 8u * (uint32_t)half);
      __syncwarp();
    };
    if (warp == 0) issue(0);
    for (int bi = 0; bi < nbatch; ++bi) {
      const int t0 = bi * TILES_PER_BATCH, nt = min(TILES_PER_BATCH, ntiles - t0), half = bi & 1;
      if (warp == 0) {
        if (bi + 1 < nbatch) issue(bi + 1);      // the other half was drained before the barrier that ended the previous iteration
        if (!mbar_wait(bar + 8u * (uint32_t)half, (parity >> half) & 1u)) { if (a.error_flag) *a.error_flag = 3; }      // one warp polls; the rest sleep in the barrier
      }
      parity ^= 1u << half;
      __syncthreads();
      tc_fence_after();
      for (int s = wg; s < nt; s += 2) {      // each warpgroup drains every second accumulator tile
        const int q = (t0 + s) * 128 + lane_row, yl = (int)__umulhi((uint32_t)q, magic_Wp), x = q - yl * Wp, y = yb + yl;
        const bool valid = yl < a.R && y < a.H && x < a.W;
        const size_t o = (((size_t)f * a.H + y) * a.W + x) * COUT;
#pragma unroll
        for (int c0 = 0; c0 < COUT; c0 += 16) {
          float v[16];
          tmem_ld16(tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)((half * TILES_PER_BATCH + s) * COUT + c0), v);
          if (!valid) continue;
          uint4 o0, o1;
          __nv_bfloat162* p0 = reinterpret_cast<__nv_bfloat162*>(&o0); __nv_bfloat162* p1 = reinterpret_cast<__nv_bfloat162*>(&o1);
#pragma unroll
          for (int i = 0; i < 16; i += 4) {
            const float4 b4 = *reinterpret_cast<const float4*>(bias_s + c0 + i);
            v[i] = fmaf(v[i], 1.0f / 255.0f, b4.x); v[i + 1] = fmaf(v[i + 1], 1.0f / 255.0f, b4.y); v[i + 2] = fmaf(v[i + 2], 1.0f / 255.0f, b4.z); v[i + 3] = fmaf(v[i + 3], 1.0f / 255.0f, b4.w);
          }
#pragma unroll
          for (int i = 0; i < 4; ++i) { p0[i] = __floats2bfloat162_rn(v[2 * i], v[2 * i + 1]); p1[i] = __floats2bfloat162_rn(v[8 + 2 * i], v[8 + 2 * i + 1]); }
          if (fused) {      // keep the band of conv outputs (already rounded to bf16, as the unfused path stores them) in shared memory
            bf16* ct = reinterpret_cast<bf16*>(xs + (size_t)a.npix_alloc * 16) + ((size_t)yl * a.W + x) * COUT + c0;
            *reinterpret_cast<uint4*>(ct) = o0; *reinterpret_cast<uint4*>(ct + 8) = o1;
          } else {
            *reinterpret_cast<uint4*>(a.out + o + c0) = o0;
            *reinterpret_cast<uint4*>(a.out + o + c0 + 8) = o1;
          }
        }
      }
      tc_fence_before();
      __syncthreads();
    }
    if (item + (int)gridDim.x < nitems) {      // loads of the next item's plane, consumed by its stage_band
      const int nitem = item + (int)gridDim.x, nf = nitem / a.nbands, nband = nitem - nf * a.nbands;
      const int nyb = fused ? max(0, 2 * nband * a.Rp - ph) : nband * a.R;
      const size_t nfr = a.frame_idx ? (size_t)a.frame_idx[nf] : (size_t)nf;
#pragma unroll
      for (int j = 0; j < 3; ++j) {
        const int i = tid + j * 256, W4 = a.W / 4, lr = i / W4, x0 = (i - lr * W4) * 4, y = nyb - 1 + lr;
        pre[j][0] = pre[j][1] = pre[j][2] = pre[j][3] = 0;
        if (i < (a.R + 2) * W4 && (unsigned)y < (unsigned)a.H)
        {
#pragma unroll
          for (int c = 0; c < 4; ++c) if (c < a.CIN) pre[j][c] = pool::ldg_early_u32(a.obs + ((nfr * a.CIN + c) * a.H + y) * a.W + x0);      // static indices: registers
        }
      }
      npre = 3;
    }
    if (fused) {
      // ---- max-pool 3x3 stride 2 SAME (A10) over the band; first maximum in row-major window order (A11) ----
      const bf16* ct = reinterpret_cast<const bf16*>(xs + (size_t)a.npix_alloc * 16);
      constexpr int C8 = COUT / 8;
      const int pr = min(a.Rp, Ho - py0);
      const uint32_t magic_Wo = (uint32_t)((0x100000000ull + (uint64_t)Wo - 1) / (uint64_t)Wo);
      for (int i = tid; i < pr * Wo * C8; i += 256) {
        const int c8 = i % C8, q = i / C8, qy = (int)__umulhi((uint32_t)q, magic_Wo), ox = q - qy * Wo, oy = py0 + qy;
        uint4 v[9]; uint32_t valid = 0;
#pragma unroll
        for (int di = 0; di < 3; ++di) {
          const int iy = oy * 2 + di - ph;
#pragma unroll
          for (int dj = 0; dj < 3; ++dj) {
            const int ix = ox * 2 + dj - pw;
            if ((unsigned)iy < (unsigned)a.H && (unsigned)ix < (unsigned)a.W) {
              v[di * 3 + dj] = *reinterpret_cast<const uint4*>(ct + ((size_t)(iy - yb) * a.W + ix) * COUT + c8 * 8);
              valid |= 1u << (di * 3 + dj);
            }
          }
        }
        const size_t o = (((size_t)f * Ho + oy) * Wo + ox) * COUT + c8 * 8;
        uint4 r; uint2 pk;
        pool::window_max(v, valid, r, pk);
        *reinterpret_cast<uint4*>(a.pool_out + o) = r;
        *reinterpret_cast<uint2*>(a.pool_arg_out + o) = pk;
      }
    }
  }
  tc_fence_before(); __syncthreads();
  if (warp == 0) tmem_dealloc(tmem_base, TMEM_COLS);
}

// stage_band with every global load of the thread issued BEFORE the first conversion (NQ quads of 4 pixels x CIN channels in registers):
// the loader warps of the warp-specialised kernel are few, so their load latency must overlap within a thread
// The same with 8-byte positions [c0 c1 c2 c3] (no constant-one channel, zero halo): the operand of the pixel-pair formulation below
template <int NQ>
__device__ __forceinline__ void stage_band8(const Args& a, uint8_t* xs, size_t fr, int yb, int tid, int nthr) {
  const int Wp = a.W + 2, W4 = a.W / 4, rows = a.R + 2, nq = rows * W4;
  const uint32_t magic_W4 = (uint32_t)((0x100000000ull + (uint64_t)W4 - 1) / (uint64_t)W4);
  for (int base = 0; base < nq; base += NQ * nthr) {
    uint32_t px[NQ][4]; int lrs[NQ], x0s[NQ];
#pragma unroll
    for (int j = 0; j < NQ; ++j) {
      const int i = base + j * nthr + tid;
      px[j][0] = px[j][1] = px[j][2] = px[j][3] = 0; lrs[j] = -1; x0s[j] = 0;
      if (i < nq) {
        const int lr = (int)__umulhi((uint32_t)i, magic_W4), x0 = (i - lr * W4) * 4, y = yb - 1 + lr;
        lrs[j] = lr; x0s[j] = x0;
        if ((unsigned)y < (unsigned)a.H) {
#pragma unroll
          for (int c = 0; c < 4; ++c) if (c < a.CIN) px[j][c] = pool::ldg_early_u32(a.obs + ((fr * a.CIN + c) * a.H + y) * a.W + x0);
        }
      }
    }
#pragma unroll
    for (int j = 0; j < NQ; ++j) {
      if (lrs[j] < 0) continue;
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const float v0 = (float)((px[j][0] >> (8 * k)) & 255u), v1 = (float)((px[j][1] >> (8 * k)) & 255u);
        const float v2 = (float)((px[j][2] >> (8 * k)) & 255u), v3 = (float)((px[j][3] >> (8 * k)) & 255u);
        __nv_bfloat162 p01 = __floats2bfloat162_rn(v0, v1), p23 = __floats2bfloat162_rn(v2, v3);
        uint2 o; o.x = *reinterpret_cast<uint32_t*>(&p01); o.y = *reinterpret_cast<uint32_t*>(&p23);
        *reinterpret_cast<uint2*>(xs + (size_t)(lrs[j] * Wp + x0s[j] + 1 + k) * 8) = o;
      }
    }
  }
  for (int i = tid; i < rows * 2; i += nthr) {       // halo columns
    int lr = i >> 1, xp = (i & 1) ? Wp - 1 : 0;
    *reinterpret_cast<uint2*>(xs + (size_t)(lr * Wp + xp) * 8) = make_uint2(0, 0);
  }
}

template <int NQ>
__device__ __forceinline__ void stage_band_batched(const Args& a, uint8_t* xs, size_t fr, int yb, int tid, int nthr) {
  const int Wp = a.W + 2, W4 = a.W / 4, rows = a.R + 2, nq = rows * W4;
  const uint32_t ONE = 0x3F80u;
  const uint32_t magic_W4 = (uint32_t)((0x100000000ull + (uint64_t)W4 - 1) / (uint64_t)W4);
  for (int base = 0; base < nq; base += NQ * nthr) {
    uint32_t px[NQ][4]; int lrs[NQ], x0s[NQ];
#pragma unroll
    for (int j = 0; j < NQ; ++j) {
      const int i = base + j * nthr + tid;
      px[j][0] = px[j][1] = px[j][2] = px[j][3] = 0; lrs[j] = -1; x0s[j] = 0;
      if (i < nq) {
        const int lr = (int)__umulhi((uint32_t)i, magic_W4), x0 = (i - lr * W4) * 4, y = yb - 1 + lr;
        lrs[j] = lr; x0s[j] = x0;
        if ((unsigned)y < (unsigned)a.H) {
#pragma unroll
          for (int c = 0; c < 4; ++c) if (c < a.CIN) px[j][c] = pool::ldg_early_u32(a.obs + ((fr * a.CIN + c) * a.H + y) * a.W + x0);
        }
      }
    }
#pragma unroll
    for (int j = 0; j < NQ; ++j) {
      if (lrs[j] < 0) continue;
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const float v0 = (float)((px[j][0] >> (8 * k)) & 255u), v1 = (float)((px[j][1] >> (8 * k)) & 255u);
        const float v2 = (float)((px[j][2] >> (8 * k)) & 255u), v3 = (float)((px[j][3] >> (8 * k)) & 255u);
        __nv_bfloat162 p01 = __floats2bfloat162_rn(v0, v1), p23 = __floats2bfloat162_rn(v2, v3);
        uint4 o; o.x = *reinterpret_cast<uint32_t*>(&p01); o.y = *reinterpret_cast<uint32_t*>(&p23); o.z = ONE; o.w = 0;
        *reinterpret_cast<uint4*>(xs + (size_t)(lrs[j] * Wp + x0s[j] + 1 + k) * 16) = o;
      }
    }
  }
  for (int i = tid; i < rows * 2; i += nthr) {       // halo columns
    int lr = i >> 1, xp = (i & 1) ? Wp - 1 : 0;
    *reinterpret_cast<uint4*>(xs + (size_t)(lr * Wp + xp) * 16) = make_uint4(0, 0, ONE, 0);
  }
}

// ------------------------------------------------------------------------------------------------
// Warp-specialised form of the fused first layer (conv 3x3 + max-pool 3x3 s2), one persistent CTA per SM.  An item is a band of Rp pooled
// rows of one frame (R = 2 Rp + 1 conv rows).
// PIXEL PAIRS: a position is 8 bytes [c0 c1 c2 c3] and an A row is the PAIR of output positions (2r, 2r+1) (Wp is even, so a pair never
// straddles an image row): for tap row di the pair needs the four input positions 2r + di Wp .. + 3 = 32 contiguous bytes = the two
// 16-byte K chunks of one K = 16 MMA (rows 16 bytes apart: LBO = 16 B, SBO = 128 B), against block-Toeplitz weights [16 x 2 Cout] (pixel e of
// the pair uses positions e .. e+2).  THREE MMAs per 256 positions instead of twelve, and a quarter of the operand bytes read from shared
// memory -- the kernel was bound by the shared-memory port (operand reads of the tensor core + epilogue stores + pool loads), not by issue.  Four roles hand items to each other through mbarriers, each two items deep, so that staging,
// tensor-core work, accumulator drain and pooling of DIFFERENT items overlap (the CTA-wide barriers of conv0_fwd_kernel serialised them):
//   warps 0-3    loaders:  uint8 frame rows -> bf16 positions of plane[s]                     PFULL[s] (4 arrivals)   <- PEMPTY[s] (MMA commit)
//   warp  4      MMA:      all tiles of the item into TMEM buffer s (256 columns each)        TFULL[s] (commit)       <- TEMPTY[s] (8 arrivals)
//   warps 5-12   epilogue: TMEM -> x 1/255 + bias -> bf16 conv band ctile[s]                  CFULL[s] (8 arrivals)   <- CEMPTY[s] (NPOOL arrivals)
//   warps 13-24  pool (the heaviest role: ~200 instructions per 8-channel window):     3x3 s2 SAME max + first arg-max (A10, A11) -> pooled map, arg-max bytes
constexpr int WS_LOAD_WARPS = 4, WS_EPI_WARPS = 8, WS_POOL_WARPS = 12, WS_THREADS = (WS_LOAD_WARPS + 1 + WS_EPI_WARPS + WS_POOL_WARPS) * 32;
struct WsArgs { Args a; uint32_t plane_bytes, ctile_bytes; };
__device__ __forceinline__ void mbar_arrive_cta(uint32_t bar) {
  asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}\n" :: "r"(bar) : "memory");
}

template <int COUT>
__global__ void __launch_bounds__(WS_THREADS, 1) conv0_fwd_ws_kernel(const WsArgs wa) {
  extern __shared__ __align__(128) uint8_t smem[];
  const Args& a = wa.a;
  constexpr uint32_t W_BYTES = 3u * 2u * (2u * COUT) * 16u;      // [di][chunk][2 Cout][8]
  __shared__ __align__(8) uint64_t bars[12];      // PFULL[2] PEMPTY[2] TFULL[2] TEMPTY[2] CFULL[2] CEMPTY[2]
  __shared__ uint32_t tmem_base_smem;
  __shared__ __align__(16) float bias_s[32];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, Wp = a.W + 2;
  const uint32_t bar0 = smem_u32(&bars[0]);
  auto PFULL = [&](int s) { return bar0 + 8u * (uint32_t)s; };        auto PEMPTY = [&](int s) { return bar0 + 8u * (uint32_t)(2 + s); };
  auto TFULL = [&](int s) { return bar0 + 8u * (uint32_t)(4 + s); };  auto TEMPTY = [&](int s) { return bar0 + 8u * (uint32_t)(6 + s); };
  auto CFULL = [&](int s) { return bar0 + 8u * (uint32_t)(8 + s); };  auto CEMPTY = [&](int s) { return bar0 + 8u * (uint32_t)(10 + s); };
  uint8_t* w_smem = smem; uint8_t* planes = smem + W_BYTES; uint8_t* ctiles = planes + 2 * (size_t)wa.plane_bytes;
  if (tid == 0) {
    for (int s = 0; s < 2; ++s) {
      mbar_init(PFULL(s), WS_LOAD_WARPS); mbar_init(PEMPTY(s), 1); mbar_init(TFULL(s), 1); mbar_init(TEMPTY(s), WS_EPI_WARPS);
      mbar_init(CFULL(s), WS_EPI_WARPS); mbar_init(CEMPTY(s), WS_POOL_WARPS);
    }
  }
  if (warp == WS_LOAD_WARPS) tmem_alloc(smem_u32(&tmem_base_smem), 512);
  for (uint32_t i = tid; i < 2 * wa.plane_bytes / 16; i += WS_THREADS) reinterpret_cast<uint4*>(planes)[i] = make_uint4(0, 0, 0, 0);
  pdl_wait(); pdl_trigger();
  if (tid < COUT) bias_s[tid] = a.bias[tid];
  for (uint32_t i = tid; i < W_BYTES / 16; i += WS_THREADS) reinterpret_cast<uint4*>(w_smem)[i] = reinterpret_cast<const uint4*>(a.w + 6 * 2 * COUT * 8)[i];      // the pair image follows the per-pixel one
  fence_async_smem();
  tc_fence_before(); __syncthreads(); tc_fence_after();
  const uint32_t tmem_base = tmem_base_smem;
  const int nitems = a.F * a.nbands;
  const int my_items = ((int)blockIdx.x < nitems) ? (nitems - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
  const int Ho = (a.H + 1) / 2, Wo = (a.W + 1) / 2;
  int th_ = (Ho - 1) * 2 + 3 - a.H; if (th_ < 0) th_ = 0; const int ph = th_ / 2;
  int tw_ = (Wo - 1) * 2 + 3 - a.W; if (tw_ < 0) tw_ = 0; const int pw = tw_ / 2;
  const int ntiles = (a.R * Wp + 255) / 256;      // 128 position pairs per tile
  auto item_geom = [&](int it, int& f, int& py0, int& yb) {
    const int item = blockIdx.x + it * gridDim.x; f = item / a.nbands; const int band = item - f * a.nbands;
    py0 = band * a.Rp; yb = max(0, 2 * py0 - ph);
  };

  if (warp < WS_LOAD_WARPS) {
    // ================= loaders =================
    for (int it = 0; it < my_items; ++it) {
      const int s = it & 1, use = it >> 1; int f, py0, yb; item_geom(it, f, py0, yb);
      if (use > 0 && !mbar_wait(PEMPTY(s), (uint32_t)((use - 1) & 1))) { if (a.error_flag) *a.error_flag = 3; }
      const size_t fr = a.frame_idx ? (size_t)a.frame_idx[f] : (size_t)f;
      stage_band8<5>(a, planes + (size_t)s * wa.plane_bytes, fr, yb, tid, WS_LOAD_WARPS * 32);
      fence_async_smem();
      __syncwarp();
      if (lane == 0) mbar_arrive_cta(PFULL(s));
    }
  } else if (warp == WS_LOAD_WARPS) {
    // ================= MMA issuer =================
    const uint32_t idesc = make_idesc(128, 2 * COUT, 0, 0);
    const uint32_t b_lo = ((smem_u32(w_smem) >> 4) & 0x3FFFu) | ((uint32_t)(2 * COUT) << 16), hi = 8u | (1u << 14);   // B: LBO 2 Cout * 16 B, SBO 128 B;  A: LBO 16 B, SBO 128 B
    for (int it = 0; it < my_items; ++it) {
      const int s = it & 1, use = it >> 1;
      if (!mbar_wait(PFULL(s), (uint32_t)(use & 1))) { if (a.error_flag) *a.error_flag = 3; }
      if (use > 0 && !mbar_wait(TEMPTY(s), (uint32_t)((use - 1) & 1))) { if (a.error_flag) *a.error_flag = 3; }
      tc_fence_after();
      const uint32_t a_lo = (((smem_u32(planes) + (uint32_t)s * wa.plane_bytes) >> 4) & 0x3FFFu) | (1u << 16);
      for (int t = 0; t < ntiles; ++t) {
        const uint32_t td = tmem_base + (uint32_t)(s * 256 + t * 2 * COUT);
#pragma unroll
        for (int di = 0; di < 3; ++di) {
          const uint32_t pos = (uint32_t)(t * 256 + di * Wp);                  // first input position of the tile's first pair: even, so pos * 8 bytes is a multiple of 16
          const uint64_t ad = ((uint64_t)hi << 32) | (uint64_t)(a_lo + (pos >> 1));
          const uint64_t bd = ((uint64_t)hi << 32) | (uint64_t)(b_lo + (uint32_t)di * 2u * (2u * COUT));
          if (elect_one()) mma_f16(td, ad, bd, idesc, di ? 1u : 0u);
        }
      }
      if (elect_one()) { mma_commit(TFULL(s)); mma_commit(PEMPTY(s)); }
      __syncwarp();
    }
  } else if (warp < WS_LOAD_WARPS + 1 + WS_EPI_WARPS) {
    // ================= epilogue: warp e drains lanes 32 (e % 4) .. +31 of every second tile =================
    const int e = warp - (WS_LOAD_WARPS + 1), q4 = warp & 3, half = e >> 2;      // TMEM lane quarter = warp index % 4 (hardware rule)
    const uint32_t magic_Wp = (uint32_t)((0x100000000ull + (uint64_t)Wp - 1) / (uint64_t)Wp);
    for (int it = 0; it < my_items; ++it) {
      const int s = it & 1, use = it >> 1; int f, py0, yb; item_geom(it, f, py0, yb);
      if (!mbar_wait(TFULL(s), (uint32_t)(use & 1))) { if (a.error_flag) *a.error_flag = 3; }
      if (use > 0 && !mbar_wait(CEMPTY(s), (uint32_t)((use - 1) & 1))) { if (a.error_flag) *a.error_flag = 3; }
      tc_fence_after();
      bf16* ct = reinterpret_cast<bf16*>(ctiles + (size_t)s * wa.ctile_bytes);
      for (int t = half; t < ntiles; t += 2) {
        const int q = t * 256 + 2 * (q4 * 32 + lane), yl = (int)__umulhi((uint32_t)q, magic_Wp), x = q - yl * Wp, y = yb + yl;      // the pair (q, q+1): same image row
        const bool rowok = yl < a.R && y < a.H;
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const bool valid = rowok && x + e < a.W;
#pragma unroll
          for (int c0 = 0; c0 < COUT; c0 += 16) {
            float v[16];
            tmem_ld16(tmem_base + ((uint32_t)(q4 * 32) << 16) + (uint32_t)(s * 256 + t * 2 * COUT + e * COUT + c0), v);
            if (!valid) continue;
            uint4 o0, o1;
            __nv_bfloat162* p0 = reinterpret_cast<__nv_bfloat162*>(&o0); __nv_bfloat162* p1 = reinterpret_cast<__nv_bfloat162*>(&o1);
#pragma unroll
            for (int i = 0; i < 16; i += 4) {
              const float4 b4 = *reinterpret_cast<const float4*>(bias_s + c0 + i);
              v[i] = fmaf(v[i], 1.0f / 255.0f, b4.x); v[i + 1] = fmaf(v[i + 1], 1.0f / 255.0f, b4.y); v[i + 2] = fmaf(v[i + 2], 1.0f / 255.0f, b4.z); v[i + 3] = fmaf(v[i + 3], 1.0f / 255.0f, b4.w);
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) { p0[i] = __floats2bfloat162_rn(v[2 * i], v[2 * i + 1]); p1[i] = __floats2bfloat162_rn(v[8 + 2 * i], v[8 + 2 * i + 1]); }
            const uint32_t off = (uint32_t)(((yl * a.W + x + e) * COUT + c0) * 2);
            *reinterpret_cast<uint4*>(reinterpret_cast<uint8_t*>(ct) + pool::ct_swz<COUT>(off)) = o0;
            *reinterpret_cast<uint4*>(reinterpret_cast<uint8_t*>(ct) + pool::ct_swz<COUT>(off + 16)) = o1;
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) { mbar_arrive_cta(TEMPTY(s)); mbar_arrive_cta(CFULL(s)); }
    }
  } else {
    // ================= pool =================
    const int pt = tid - (WS_LOAD_WARPS + 1 + WS_EPI_WARPS) * 32;
    constexpr int NP = WS_POOL_WARPS * 32;
    for (int it = 0; it < my_items; ++it) {
      const int s = it & 1, use = it >> 1; int f, py0, yb; item_geom(it, f, py0, yb);
      if (!mbar_wait(CFULL(s), (uint32_t)(use & 1))) { if (a.error_flag) *a.error_flag = 3; }
      pool::pool_band<COUT>(ctiles + (size_t)s * wa.ctile_bytes, yb, py0, min(a.Rp, Ho - py0), f, a.H, a.W, Ho, Wo, ph, pw, a.pool_out, a.pool_arg_out, pt, NP);
      __syncwarp();
      if (lane == 0) mbar_arrive_cta(CEMPTY(s));
    }
  }
  tc_fence_before(); __syncthreads();
  if (warp == WS_LOAD_WARPS) tmem_dealloc(tmem_base, 512);
}

__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}\n" :: "r"(bar) : "memory");
}

constexpr int WNLOAD = 512;     // warps 0-15 stage (the gather is latency-bound: more loads in flight); warps 0-1 later drain TMEM; warp 16 issues the MMAs

// Two stages of (X plane, DY region): the loaders fill one while the tensor core reads the other.  ONE MMA [64 x 3*COUT] per
// 16 positions: the A descriptor walks M over neighbouring positions (rows 8*dj + c), the B descriptor walks N over image rows
// of the swizzled DY region (column group e pairs with the tap row di = 2 - e; see wgrad_tc.cu).  Accumulator row r sits in
// TMEM lane 32*(r/16) + r%16.
template <int COUT>
__global__ void __launch_bounds__(WNLOAD + 32) conv0_wgrad_kernel(const Args a) {
  extern __shared__ __align__(128) uint8_t smem_raw[];
  constexpr int YCH = COUT / 8;
  constexpr uint32_t TCOLS = 128, PY = 2u * COUT, SWY = COUT == 16 ? 6u : 4u;
  __shared__ __align__(8) uint64_t bars[5];       // full[2], empty[2], done
  __shared__ uint32_t tmem_base_smem;
  const int tid = threadIdx.x, warp = tid >> 5, Wp = a.W + 2;
  uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  const uint32_t XB = (((uint32_t)(a.w_xoff + a.npix_alloc) * 16u) + 1023u) & ~1023u, STAGE = XB + (uint32_t)a.w_ybytes;
  const uint32_t bar0 = smem_u32(&bars[0]);
  if (tid == 0) {
    for (int i = 0; i < 5; ++i) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" :: "r"(bar0 + 8u * i) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  if (warp == WNLOAD / 32) tmem_alloc(smem_u32(&tmem_base_smem), TCOLS);
  for (int st = 0; st < 2; ++st) {
    uint8_t* xs = smem + (size_t)st * STAGE;
    for (uint32_t i = tid; i < XB / 16; i += WNLOAD + 32) reinterpret_cast<uint4*>(xs)[i] = make_uint4(0, 0, 0x3F80u, 0);
    for (uint32_t i = tid; i < (uint32_t)a.w_ybytes / 16; i += WNLOAD + 32) reinterpret_cast<uint4*>(xs + XB)[i] = make_uint4(0, 0, 0, 0);
  }
  pdl_wait(); pdl_trigger();      // the prologue above is private to the CTA (tc_ptx.cuh)
  fence_async_smem();
  tc_fence_before(); __syncthreads(); tc_fence_after();
  const uint32_t tmem_base = tmem_base_smem;
  const int nitems = a.F * a.nbands;
  const int my_items = ((int)blockIdx.x < nitems) ? (nitems - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
  if (warp < WNLOAD / 32) {
    // two loader teams of eight warps; team t stages the items it = t, t+2, ... into stage t, so the global-load latencies and the
    // barrier chains of two consecutive items overlap
    constexpr int TN = WNLOAD / 2;
    const int team = tid / TN, ttid = tid - team * TN;
    for (int it = team; it < my_items; it += 2) {
      const int item = blockIdx.x + it * gridDim.x, s = team, use = it >> 1;
      const int f = item / a.nbands, yb = (item - f * a.nbands) * a.R;
      // the pooled gradients of this thread's first item of each phase are fetched before anything waits
      PoolGeom q; bool pf_ok[4] = {false, false, false, false}; int pf_oy[4], pf_ox[4], pf_ch[4]; uint2 pf_pk[4]; uint4 pf_dv[4];
      if (a.pool_arg != nullptr) {
        q = pool_geom(a, yb);
#pragma unroll
        for (int p = 0; p < 4; ++p) {
          pf_ok[p] = pool_item(q, p, ttid, YCH, pf_oy[p], pf_ox[p], pf_ch[p]);
          if (pf_ok[p]) {
            const size_t o = (((size_t)f * q.Ho + pf_oy[p]) * q.Wo + pf_ox[p]) * COUT + pf_ch[p] * 8;
            pf_pk[p] = pool::ldg_early_v2(a.pool_arg + o); pf_dv[p] = pool::ldg_early_v4(a.dpool + o);
          }
        }
      }
      const size_t fr = a.frame_idx ? (size_t)a.frame_idx[f] : (size_t)f;
      uint32_t pre[2][4];      // this thread's first two observation quads, also fetched ahead of the wait
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const int i = ttid + j * TN, W4 = a.W / 4, lr = i / W4, x0 = (i - lr * W4) * 4, y = yb - 1 + lr;
        pre[j][0] = pre[j][1] = pre[j][2] = pre[j][3] = 0;
        if (i < (a.R + 2) * W4 && (unsigned)y < (unsigned)a.H)
          for (int c = 0; c < a.CIN; ++c) pre[j][c] = pool::ldg_early_u32(a.obs + ((fr * a.CIN + c) * a.H + y) * a.W + x0);
      }
      if (use > 0 && !mbar_wait(bar0 + 8u * (2 + s), (uint32_t)((use - 1) & 1))) { if (a.error_flag) *a.error_flag = 4; }
      uint8_t* xs = smem + (size_t)s * STAGE + (size_t)a.w_xoff * 16; uint8_t* ys = smem + (size_t)s * STAGE + XB + (size_t)a.w_yoff * PY;
      const uint32_t ys_addr = smem_u32(ys);
      stage_band(a, xs, fr, yb, ttid, TN, pre, 2);
      if (a.pool_arg == nullptr) {
        for (int i = ttid; i < a.kext * YCH; i += TN) {
          int ch = i % YCH, pos = i / YCH, yl = pos / Wp, x = pos - yl * Wp, y = yb + yl;
          uint4 v = make_uint4(0, 0, 0, 0);
          if (yl < a.R && y < a.H && x < a.W) v = *reinterpret_cast<const uint4*>(a.dy + (((size_t)f * a.H + y) * a.W + x) * COUT + ch * 8);
          *reinterpret_cast<uint4*>(dy_chunk<COUT>(ys, ys_addr, pos, ch)) = v;
        }
      } else {
        for (int i = ttid; i < a.kext * YCH; i += TN)
          reinterpret_cast<uint4*>(ys)[i] = make_uint4(0, 0, 0, 0);
#pragma unroll
        for (int p = 0; p < 4; ++p) {
          asm volatile("bar.sync %0, %1;\n" :: "r"(1 + team), "n"(TN) : "memory");
          if (pf_ok[p]) pool_scatter<COUT>(a, q, ys, ys_addr, yb, pf_oy[p], pf_ox[p], pf_ch[p], pf_pk[p], pf_dv[p]);
          for (int i = ttid + TN; ; i += TN) {
            int oy, ox, ch; if (!pool_item(q, p, i, YCH, oy, ox, ch)) break;
            const size_t o = (((size_t)f * q.Ho + oy) * q.Wo + ox) * COUT + ch * 8;
            pool_scatter<COUT>(a, q, ys, ys_addr, yb, oy, ox, ch, *reinterpret_cast<const uint2*>(a.pool_arg + o), *reinterpret_cast<const uint4*>(a.dpool + o));
          }
        }
      }
      fence_async_smem();
      asm volatile("bar.sync %0, %1;\n" :: "r"(1 + team), "n"(TN) : "memory");
      if (ttid == 0) mbar_arrive(bar0 + 8u * s);
    }
    if (warp < 2) {
      if (my_items > 0 && !mbar_wait(bar0 + 8u * 4, 0u)) { if (a.error_flag) *a.error_flag = 4; }
      tc_fence_after();
      float* out = a.partial + (size_t)blockIdx.x * 3 * 24 * COUT;
      const int lane = tid & 31, row = lane < 16 ? warp * 16 + lane : 1 << 20;
      for (int di = 0; di < 3; ++di) {
#pragma unroll
        for (int c0 = 0; c0 < COUT; c0 += 16) {
          float v[16];
          tmem_ld16(tmem_base + ((uint32_t)(warp * 32) << 16) + (uint32_t)(di * COUT + c0), v);
          if (row < 24) {
#pragma unroll
            for (int i = 0; i < 16; ++i) out[((size_t)(2 - di) * 24 + row) * COUT + c0 + i] = v[i];      // column group e = di holds the tap row 2 - e
          }
        }
      }
    }
  } else {      // warp WNLOAD / 32: the whole warp runs the loop, one elected lane issues
    const uint32_t idesc = make_idesc(64, 3 * COUT, 1, 1);
    const uint32_t a_hi = 1u | (1u << 14), b_hi = ((8u * PY) >> 4) | (1u << 14) | (SWY << 29);     // A: SBO = 16 B (M walk); B: SBO = 8 rows, swizzled
    const int r_begin = ((a.w_yoff - 2 * Wp) / 16) * 16, r_end = a.kext + a.w_yoff;               // stored DY rows the contraction runs over
    uint32_t accumulate = 0;
    for (int it = 0; it < my_items; ++it) {
      const int s = it & 1, use = it >> 1;
      if (!mbar_wait(bar0 + 8u * s, (uint32_t)(use & 1))) { if (a.error_flag) *a.error_flag = 4; }
      tc_fence_after();
      const uint32_t x_base = smem_u32(smem + (size_t)s * STAGE), y_base = x_base + XB;
      uint32_t xl = (((x_base >> 4) & 0x3FFFu) | (8u << 16)) + (uint32_t)(a.w_xoff + r_begin - (a.w_yoff - 2 * Wp));      // LBO = 128 B; 16 B per position
      uint32_t yl = (((y_base >> 4) & 0x3FFFu) | ((((uint32_t)Wp * PY) >> 4) << 16)) + (uint32_t)r_begin * (PY >> 4);  // LBO = one image row
#pragma unroll 4
      for (int r = r_begin; r < r_end; r += 16) {
        if (elect_one()) mma_f16(tmem_base, ((uint64_t)a_hi << 32) | xl, ((uint64_t)b_hi << 32) | yl, idesc, accumulate);
        accumulate = 1;
        xl += 16u; yl += PY;
      }
      if (elect_one()) mma_commit(bar0 + 8u * (2 + s));
      __syncwarp();
    }
    if (elect_one()) mma_commit(bar0 + 8u * 4);
    __syncwarp();
  }
  tc_fence_before(); __syncthreads();
  if (warp == WNLOAD / 32) tmem_dealloc(tmem_base, TCOLS);
}

// forward B image: slot = 2*di + h; h = 0: chunks (di,0),(di,1); h = 1: chunks (di,2), zero.  [slot][chunk][o][8]
__global__ void conv0_pack_kernel(const float* __restrict__ params, Geom g, ParamMap pm, bf16* __restrict__ wimg) {
  int total = 6 * 2 * g.Cout * 8;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < total; i += gridDim.x * blockDim.x) {
    int c = i & 7, o = (i >> 3) % g.Cout, chunk = ((i >> 3) / g.Cout) & 1, slot = (i >> 3) / g.Cout / 2;
    int di = slot >> 1, dj = (slot & 1) * 2 + chunk;
    float v = (c < g.Cin && dj < 3) ? params[pm.w(o, c, di, dj, g)] : 0.f;
    wimg[i] = __float2bfloat16_rn(v);
  }
}

__global__ void conv0_wgrad_reduce_kernel(const float* __restrict__ partial, int nctas, Geom g, ParamMap pm, float* __restrict__ grad) {
  const int per = 3 * 24 * g.Cout;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < per; i += gridDim.x * blockDim.x) {
    float s = 0.f;
    int z = 0;
    for (; z + 16 <= nctas; z += 16) {      // 16 loads in flight, then the additions in CTA order
      float v[16];
#pragma unroll
      for (int k = 0; k < 16; ++k) v[k] = __ldg(partial + (size_t)(z + k) * per + i);
#pragma unroll
      for (int k = 0; k < 16; ++k) s += v[k];
    }
    for (; z < nctas; ++z) s += partial[(size_t)z * per + i];
    int o = i % g.Cout, row = (i / g.Cout) % 24, di = i / g.Cout / 24, dj = row >> 3, c = row & 7;
    if (c < g.Cin) grad[pm.w(o, c, di, dj, g)] = s * (1.0f / 255.0f);
    else if (c == 4 && dj == 0 && di == 0) grad[pm.b(o)] = s;
  }
}

}  // namespace tc0

bool conv0_tc_supported(const Geom& g) {
  return g.kh == 3 && g.kw == 3 && g.s == 1 && g.p == 1 && g.Cin <= 4 && (g.Cout == 16 || g.Cout == 32) && g.W % 4 == 0 && g.W >= 8 && g.H == g.Ho && g.W == g.Wo;
}
constexpr int CONV0_MAX_CTAS = 148;
size_t conv0_partial_elems(const Geom& g) { return (size_t)CONV0_MAX_CTAS * 3 * 24 * g.Cout; }
size_t conv0_wimg_elems(const Geom& g) { return (size_t)2 * 6 * 2 * g.Cout * 8; }      // two images of 96 Cout elements: [6][2][Cout][8] (one pixel per row) and [3][2][2 Cout][8] (pixel pairs)

int launch_conv0_pack(const Geom& g, const ParamMap& pm, const float* params, bf16* wimg, cudaStream_t st) {
  tc0::conv0_pack_kernel<<<(6 * 2 * g.Cout * 8 + 255) / 256, 256, 0, st>>>(params, g, pm, wimg);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

template <class K>
static int set_smem(K kernel, size_t smem, size_t*) { return ensure_dyn_smem((const void*)kernel, smem); }

int launch_conv0_fwd(const Geom& g, int F, const uint8_t* obs, const int32_t* frame_idx, const bf16* wimg, const float* bias, bf16* out,
                     bf16* pool_out, uint8_t* pool_arg, int* error_flag, cudaStream_t st) {
  if (F <= 0) return CB_OK;
  const int Wp = g.W + 2;
  int R, nb, Rp = 0; size_t ctile = 0;
  if (pool_out) {      // fused max-pool: a band of Rp pooled rows needs 2 Rp + 1 conv rows, kept in shared memory as bf16
    const int Ho = (g.H + 1) / 2;
    auto need = [&](int rp) { const int r = 2 * rp + 1; return (size_t)6 * 2 * g.Cout * 16 + (size_t)(((r * Wp + 127) / 128) * 128 + 2 * Wp + 8) * 16 + (size_t)r * g.W * g.Cout * 2; };
    Rp = 1; while (Rp < Ho && need(Rp + 1) <= (size_t)110 * 1024) ++Rp;      // two CTAs per SM
    nb = (Ho + Rp - 1) / Rp; Rp = (Ho + nb - 1) / nb;                          // equal bands
    R = 2 * Rp + 1;
    ctile = (size_t)R * g.W * g.Cout * 2;
  } else {
    R = std::min(g.H, (90 * 1024 / 16 - 2 * Wp - 130) / Wp - 2); if (R < 1) R = 1;
    nb = (g.H + R - 1) / R; R = (g.H + nb - 1) / nb;
  }
  if (pool_out) {
    // warp-specialised kernel: bands of Rp pooled rows whose tiles fit one 256-column TMEM buffer, two planes + two conv bands in shared memory
    const int Ho = (g.H + 1) / 2;
    auto tiles_of = [&](int rp) { return ((2 * rp + 1) * Wp + 255) / 256; };      // 128 position pairs per tile
    auto npix_of = [&](int rp) { return (tiles_of(rp) * 256 + 2 * Wp + 16 + 15) / 16 * 16; };        // 8-byte positions (a multiple of 128 bytes); the last tile's MMAs read up to 2 Wp + 3 positions further
    auto smem_of = [&](int rp) { return (size_t)3 * 2 * 2 * g.Cout * 16 + 2 * (size_t)npix_of(rp) * 8 + 2 * (size_t)(2 * rp + 1) * g.W * g.Cout * 2; };
    int rp = 1; while (rp < Ho && tiles_of(rp + 1) * 2 * g.Cout <= 256 && smem_of(rp + 1) <= (size_t)200 * 1024) ++rp;
    if (Wp % 2 == 0 && tiles_of(rp) * 2 * g.Cout <= 256 && smem_of(rp) <= (size_t)200 * 1024) {
      const int nbw = (Ho + rp - 1) / rp; rp = (Ho + nbw - 1) / nbw;      // equal bands
      const int Rw = 2 * rp + 1, npw = npix_of(rp);
      tc0::WsArgs wa{{obs, frame_idx, wimg, bias, out, nullptr, nullptr, nullptr, nullptr, F, g.H, g.W, g.Cin, Rw, nbw, npw, 0, 0, 0, 0, pool_out, pool_arg, rp, error_flag},
                     (uint32_t)npw * 8u, (uint32_t)((size_t)Rw * g.W * g.Cout * 2)};
      const int gridw = std::min(F * nbw, 148); int rcw;
      if (g.Cout == 16) { if ((rcw = ensure_dyn_smem((const void*)tc0::conv0_fwd_ws_kernel<16>, smem_of(rp)))) return rcw; CB_CUDA(launch_pdl(tc0::conv0_fwd_ws_kernel<16>, dim3(gridw), dim3(tc0::WS_THREADS), smem_of(rp), st, wa)); }
      else { if ((rcw = ensure_dyn_smem((const void*)tc0::conv0_fwd_ws_kernel<32>, smem_of(rp)))) return rcw; CB_CUDA(launch_pdl(tc0::conv0_fwd_ws_kernel<32>, dim3(gridw), dim3(tc0::WS_THREADS), smem_of(rp), st, wa)); }
      CB_CUDA(cudaGetLastError());
      return CB_OK;
    }
  }
  const int npix = ((R * Wp + 127) / 128) * 128 + 2 * Wp + 8;
  const size_t smem = (size_t)6 * 2 * g.Cout * 16 + (size_t)npix * 16 + ctile;
  tc0::Args a{obs, frame_idx, wimg, bias, out, nullptr, nullptr, nullptr, nullptr, F, g.H, g.W, g.Cin, R, nb, npix, 0, 0, 0, 0, pool_out, pool_arg, Rp, error_flag};
  const int grid = std::min(F * nb, 296);
  static size_t c16 = 0, c32 = 0; int rc;
  if (g.Cout == 16) { if ((rc = set_smem(tc0::conv0_fwd_kernel<16>, smem, &c16))) return rc; tc0::conv0_fwd_kernel<16><<<grid, 256, smem, st>>>(a); }
  else { if ((rc = set_smem(tc0::conv0_fwd_kernel<32>, smem, &c32))) return rc; tc0::conv0_fwd_kernel<32><<<grid, 256, smem, st>>>(a); }
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

int launch_conv0_wgrad(const Geom& g, const ParamMap& pm, int F, const uint8_t* obs, const int32_t* frame_idx, const bf16* dy, const uint8_t* pool_arg,
                       const bf16* dpool, float* partial, float* grad, int* error_flag, cudaStream_t st) {
  if (F <= 0) return CB_OK;
  const int Wp = g.W + 2, py = 2 * g.Cout;
  const int xoff = 16, per = 1024 / py, yoff = (2 * Wp + per - 1) / per * per;      // the swizzled DY rows start on a 1024-byte boundary
  auto a1k = [](size_t b) { return (b + 1023) & ~(size_t)1023; };
  auto plan = [&](int R, int* kext, int* npix, size_t* ybytes) {      // bytes of one stage (X plane + DY region) for bands of R rows
    *kext = (R * Wp + 15) / 16 * 16; *npix = (*kext + 2 * Wp + 40 + 7) / 8 * 8;
    *ybytes = a1k((size_t)(yoff + *npix) * py);
    return a1k((size_t)(xoff + *npix) * 16) + *ybytes;
  };
  int kext, npix; size_t ybytes;
  int R = g.H; while (R > 1 && 2 * plan(R, &kext, &npix, &ybytes) + 1024 > (size_t)200 * 1024) --R;
  const int nb = (g.H + R - 1) / R; R = (g.H + nb - 1) / nb;
  const size_t smem = 2 * plan(R, &kext, &npix, &ybytes) + 1024;
  const int grid = std::min(F * nb, CONV0_MAX_CTAS);
  tc0::Args a{obs, frame_idx, nullptr, nullptr, nullptr, dy, partial, pool_arg, dpool, F, g.H, g.W, g.Cin, R, nb, npix, kext, xoff, yoff, (int)ybytes,
              nullptr, nullptr, 0, error_flag};
  static size_t c16 = 0, c32 = 0; int rc;
  if (g.Cout == 16) { if ((rc = set_smem(tc0::conv0_wgrad_kernel<16>, smem, &c16))) return rc; CB_CUDA(launch_pdl(tc0::conv0_wgrad_kernel<16>, dim3(grid), dim3(tc0::WNLOAD + 32), smem, st, a)); }
  else { if ((rc = set_smem(tc0::conv0_wgrad_kernel<32>, smem, &c32))) return rc; CB_CUDA(launch_pdl(tc0::conv0_wgrad_kernel<32>, dim3(grid), dim3(tc0::WNLOAD + 32), smem, st, a)); }
  CB_CUDA(cudaGetLastError());
  tc0::conv0_wgrad_reduce_kernel<<<(3 * 24 * g.Cout + 255) / 256, 256, 0, st>>>(partial, grid, g, pm, grad);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

}  // namespace cb
