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
