// TMA (cp.async.bulk.tensor) helpers: a 4-D tiled tensor map over an NHWC bf16 activation tensor whose box is
// [8 channels][box_w][box_h][box_f].  With the box started at (x, y) = (-1, -1) the out-of-bounds elements are
// zero-filled by the hardware, so ONE bulk copy per 8-channel chunk lands a group of frames in shared memory
// exactly in the pixel-linear plane layout of conv_tc.cu / wgrad_tc.cu, zero halo included.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdlib.h>

namespace cb {
namespace tma {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// CB_DISABLE_TMA=1 in the environment makes every tensor-map request fail, which selects the kernels that stage their operands through
// the load/store units (conv3x3_tc_kernel, wgrad3x3_tc_kernel; the fc layer falls back to the SIMT GEMM): the paths a driver without
// cuTensorMapEncodeTiled would take.  tests/test_gpu_learner.py::test_no_tma_fallback_kernels runs them under the oracle.
inline EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  static const bool disabled = [] { const char* e = getenv("CB_DISABLE_TMA"); return e && e[0] == '1'; }();
  if (disabled) return nullptr;
  if (!fn) {
    void* p = nullptr; cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess) fn = (EncodeTiledFn)p;
  }
  return fn;
}

// tensor [F][H][W][C] bf16 (C fastest); returns false if the driver refuses the map.
// box_c = 8: one 8-channel chunk per copy (plane layout, 16-byte pieces).  box_c = C in {16, 32, 64} with swizzle = true: whole
// pixels (32/64/128-byte pieces: the TMA unit moves about one piece per clock whatever its size) written in the 32B/64B/128B
// swizzle pattern, i.e. the canonical swizzled UMMA layout with one shared-memory row per pixel.
inline bool make_nhwc_map(CUtensorMap* m, const void* base, int F, int H, int W, int C, int box_w, int box_h, int box_f, int box_c = 8, bool swizzle = false) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return false;
  cuuint64_t dims[4] = {(cuuint64_t)C, (cuuint64_t)W, (cuuint64_t)H, (cuuint64_t)F};
  cuuint64_t strides[3] = {(cuuint64_t)C * 2, (cuuint64_t)W * C * 2, (cuuint64_t)H * W * C * 2};
  cuuint32_t box[4] = {(cuuint32_t)box_c, (cuuint32_t)box_w, (cuuint32_t)box_h, (cuuint32_t)box_f};
  cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
  CUtensorMapSwizzle sw = CU_TENSOR_MAP_SWIZZLE_NONE;
  if (swizzle) sw = box_c == 16 ? CU_TENSOR_MAP_SWIZZLE_32B : (box_c == 32 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_128B);
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            sw, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// 2-D row-major bf16 matrix [rows][cols] (cols contiguous, cols * 2 bytes a multiple of 16); box = box_rows x box_cols with the 128-byte
// swizzle when box_cols = 64.  Out-of-range parts of a box are zero-filled.
inline bool make_2d_map(CUtensorMap* m, const void* base, int rows, int cols, int box_rows, int box_cols) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
  cuuint64_t strides[1] = {(cuuint64_t)cols * 2};
  cuuint32_t box[2] = {(cuuint32_t)box_cols, (cuuint32_t)box_rows};
  cuuint32_t estr[2] = {1u, 1u};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            box_cols == 64 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

__device__ __forceinline__ void arrive_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void load_4d(uint32_t dst_smem, const CUtensorMap* map, int c0, int x, int y, int f, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];\n"
               :: "r"(dst_smem), "l"((uint64_t)map), "r"(c0), "r"(x), "r"(y), "r"(f), "r"(bar) : "memory");
}
__device__ __forceinline__ void prefetch_map(const CUtensorMap* map) {
  asm volatile("prefetch.tensormap [%0];\n" :: "l"((uint64_t)map) : "memory");
}

}  // namespace tma
}  // namespace cb
