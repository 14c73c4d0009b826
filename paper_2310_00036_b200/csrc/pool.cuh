// Device helpers for the 3x3 stride-2 SAME max-pool (A10) on packed bf16 channel vectors (8 channels = 16 B).
#pragma once
#include <cuda_bf16.h>
#include <stdint.h>

namespace cb {
namespace pool {

// Maximum over the valid taps of a window (bit t of `valid` = tap t = 3*di + dj holds data in v[t]) and, per
// channel, the position of the FIRST maximum in row-major window order (A11).  Packed bf16x2 arithmetic: a max
// pass, then an equality pass from the last tap to the first so that the earliest equal tap wins.  One byte of
// `arg` per channel.
__device__ __forceinline__ void window_max(const uint4 (&v)[9], uint32_t valid, uint4& best, uint2& arg) {
  __nv_bfloat162 m[4];
  const uint32_t NEG_INF2 = 0xFF80FF80u;
  if (valid == 0x1FFu) {      // interior window (all but the border ones): no per-tap predicates
    const __nv_bfloat162* h0 = reinterpret_cast<const __nv_bfloat162*>(&v[0]);
#pragma unroll
    for (int k = 0; k < 4; ++k) m[k] = h0[k];
#pragma unroll
    for (int t = 1; t < 9; ++t) {
      const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&v[t]);
#pragma unroll
      for (int k = 0; k < 4; ++k) m[k] = __hmax2(m[k], h[k]);
    }
    uint32_t a[4] = {0x00080008u, 0x00080008u, 0x00080008u, 0x00080008u};      // tap 8 equals the maximum unless an earlier one does
#pragma unroll
    for (int t = 7; t >= 0; --t) {
      const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&v[t]);
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const uint32_t mask = __heq2_mask(h[k], m[k]);
        a[k] = (a[k] & ~mask) | (((uint32_t)t * 0x00010001u) & mask);
      }
    }
    best.x = *reinterpret_cast<const uint32_t*>(&m[0]); best.y = *reinterpret_cast<const uint32_t*>(&m[1]);
    best.z = *reinterpret_cast<const uint32_t*>(&m[2]); best.w = *reinterpret_cast<const uint32_t*>(&m[3]);
    arg.x = __byte_perm(a[0], a[1], 0x6420); arg.y = __byte_perm(a[2], a[3], 0x6420);
    return;
  }
#pragma unroll
  for (int k = 0; k < 4; ++k) m[k] = *reinterpret_cast<const __nv_bfloat162*>(&NEG_INF2);
#pragma unroll
  for (int t = 0; t < 9; ++t)
    if ((valid >> t) & 1u) {
      const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&v[t]);
#pragma unroll
      for (int k = 0; k < 4; ++k) m[k] = __hmax2(m[k], h[k]);
    }
  uint32_t a[4] = {0x000F000Fu, 0x000F000Fu, 0x000F000Fu, 0x000F000Fu};
#pragma unroll
  for (int t = 8; t >= 0; --t)
    if ((valid >> t) & 1u) {
      const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&v[t]);
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const uint32_t mask = __heq2_mask(h[k], m[k]);
        a[k] = (a[k] & ~mask) | (((uint32_t)t * 0x00010001u) & mask);
      }
    }
  best.x = *reinterpret_cast<const uint32_t*>(&m[0]); best.y = *reinterpret_cast<const uint32_t*>(&m[1]);
  best.z = *reinterpret_cast<const uint32_t*>(&m[2]); best.w = *reinterpret_cast<const uint32_t*>(&m[3]);
  arg.x = __byte_perm(a[0], a[1], 0x6420); arg.y = __byte_perm(a[2], a[3], 0x6420);
}

// Bank-conflict-free layout of a conv band kept in shared memory as [row][x][channel] bf16: inside every 64-byte block (a pixel pair at 16
// channels, one pixel at 32, half a pixel at 64) the 16-byte chunk c sits at c ^ f((block >> 1) & 3).  The lanes of a TMEM-draining warp (64 /
// 128 bytes apart) and the lanes of a pooling warp (one or two pixels apart) then spread over all eight 16-byte bank groups.  At 16 channels
// f must swap the two bits (neighbouring pool lanes are ONE block apart); from 32 channels on the identity does (two shift/logic instructions).
template <int COUT>
__device__ __forceinline__ uint32_t ct_swz(uint32_t byte_off) {
  if (COUT == 16) return byte_off ^ (((byte_off >> 2) & 0x20u) | ((byte_off >> 4) & 0x10u));
  return byte_off ^ ((byte_off >> 3) & 0x30u);
}

// 3x3 stride-2 SAME max-pool (A10) with first arg-max (A11) over `pr` pooled rows starting at row py0 of frame f, read from the swizzled conv
// band `ctb` whose first row is conv row yb.  Thread pt of NP; writes the pooled map and the arg-max bytes.
template <int COUT>
__device__ __forceinline__ void pool_band(const uint8_t* ctb, int yb, int py0, int pr, int f, int H, int W, int Ho, int Wo, int ph, int pw,
                                          __nv_bfloat16* __restrict__ pool_out, uint8_t* __restrict__ pool_arg, int pt, int NP) {
  constexpr int C8 = COUT / 8, LC8 = COUT == 16 ? 1 : (COUT == 32 ? 2 : 3);
  constexpr uint32_t PIX = COUT * 2;
  const uint32_t magic_Wo = (uint32_t)((0x100000000ull + (uint64_t)Wo - 1) / (uint64_t)Wo);
  const uint32_t rowp = (uint32_t)W * PIX;
  const size_t obase = (size_t)f * Ho * Wo * COUT;
  const int ntask = pr * Wo * C8;
  for (int i = pt; i < ntask; i += NP) {
    const int c8 = i & (C8 - 1), q = i >> LC8, qy = (int)__umulhi((uint32_t)q, magic_Wo), ox = q - qy * Wo, oy = py0 + qy;
    uint4 v[9]; uint32_t valid = 0;
    const int iy0 = oy * 2 - ph, ix0 = ox * 2 - pw;
    if (iy0 >= 0 && iy0 + 2 < H && ix0 >= 0 && ix0 + 2 < W) {      // interior window (all but the border ones): no per-tap predicates
      const uint32_t base = (uint32_t)((iy0 - yb) * W + ix0) * PIX + (uint32_t)c8 * 16u;
#pragma unroll
      for (int di = 0; di < 3; ++di)
#pragma unroll
        for (int dj = 0; dj < 3; ++dj) v[di * 3 + dj] = *reinterpret_cast<const uint4*>(ctb + ct_swz<COUT>(base + di * rowp + dj * PIX));
      valid = 0x1FFu;
    } else {
#pragma unroll
      for (int di = 0; di < 3; ++di) {
        const int iy = iy0 + di;
#pragma unroll
        for (int dj = 0; dj < 3; ++dj) {
          const int ix = ix0 + dj;
          if ((unsigned)iy < (unsigned)H && (unsigned)ix < (unsigned)W) {
            v[di * 3 + dj] = *reinterpret_cast<const uint4*>(ctb + ct_swz<COUT>((uint32_t)((iy - yb) * W + ix) * PIX + (uint32_t)c8 * 16u));
            valid |= 1u << (di * 3 + dj);
          }
        }
      }
    }
    const size_t o = obase + (size_t)((uint32_t)(oy * Wo + ox) * (uint32_t)COUT + (uint32_t)c8 * 8u);
    uint4 r; uint2 pk;
    window_max(v, valid, r, pk);
    *reinterpret_cast<uint4*>(pool_out + o) = r;
    *reinterpret_cast<uint2*>(pool_arg + o) = pk;
  }
}

// loads the compiler may not sink to their first use: issued where written (ahead of a barrier wait), consumed after it
__device__ __forceinline__ uint32_t ldg_early_u32(const void* p) {
  uint32_t v; asm volatile("ld.global.nc.u32 %0, [%1];\n" : "=r"(v) : "l"(p)); return v;
}
__device__ __forceinline__ uint2 ldg_early_v2(const void* p) {
  uint2 v; asm volatile("ld.global.nc.v2.u32 {%0,%1}, [%2];\n" : "=r"(v.x), "=r"(v.y) : "l"(p)); return v;
}
__device__ __forceinline__ uint4 ldg_early_v4(const void* p) {
  uint4 v; asm volatile("ld.global.nc.v4.u32 {%0,%1,%2,%3}, [%4];\n" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p)); return v;
}

// dst (one bf16) += g, rounded to bf16; plain read-modify-write (the caller orders conflicting writers)
__device__ __forceinline__ void add_bf16(uint16_t* dst, uint16_t g) {
  const float o = __uint_as_float((uint32_t)(*dst) << 16), t = __uint_as_float((uint32_t)g << 16);
  const __nv_bfloat16 r = __float2bfloat16_rn(o + t);
  *dst = *reinterpret_cast<const uint16_t*>(&r);
}

}  // namespace pool
}  // namespace cb
