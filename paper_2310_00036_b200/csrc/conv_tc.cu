// tcgen05 / TMEM implicit-GEMM 3x3 convolution (stride 1, zero pad 1) for CB_PREC_BF16_TC, sm_100a.
//
// One kernel serves the forward conv and its dgrad (the same convolution with flipped taps and
// transposed weights; only the packed weights and the epilogue differ).
//
// Data layout in shared memory: an item (G whole frames with their zero halo, or one row band of a frame) is landed by ONE 4-D
// `cp.async.bulk.tensor` whose box starts at (-1, -1): the out-of-bounds zero fill IS the conv halo.  A stage holds whole pixels, one
// row of 2*Cin bytes per position q = j*R + (y+1)*Wp + (x+1) (R = (H+2)*(W+2), Wp = W+2), in the 32B/64B/128B swizzle pattern the TMA
// unit writes and the K-major UMMA descriptor names.  For an output position q the input under tap (di,dj) is at position
// q + di*Wp + dj: a tap is a constant shift of the descriptor's start address (the swizzle is a function of the absolute address, so a
// descriptor may start at any row).  The whole 3x3 conv is 9*Cin/16 tcgen05.mma instructions per 128-position tile with the fp32
// accumulator in TMEM.  Positions that fall on halo columns/rows are computed and dropped (6-40% of the rows: the price of needing
// no im2col and no per-tap copies).  Weights: B operand [Cout x 16] per (tap, k-step), K-major canonical layout, staged once per CTA.
// Without TMA (no cuTensorMapEncodeTiled, or CB_DISABLE_TMA=1) conv_tc_supported() is false and the layer runs on the SIMT implicit GEMM.
#include "common.cuh"
#include "tma.cuh"

#include <cstring>
#include "tc_ptx.cuh"

namespace cb {

namespace tc {

using namespace ptx;      // tcgen05 / TMEM / mbarrier wrappers: tc_ptx.cuh

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

// ------------------------------------------------------------------------------------------------
// The kernel: one persistent CTA per SM, warp-specialised.
//   warp 16     TMA producer: lands item i+1.. into a ring of NS shared-memory stages
//   warps 18-21 (relu_in only) apply the ReLU in place on a landed stage, then publish it
//   warp 17     MMA issuer (one elected lane): accumulates batches of tiles into a ring of 4 TMEM buffers of 128 columns
//   warps 0-15  epilogue: four warpgroups drain every fourth tile of a finished batch while the next batch is computed
// mbarriers: raw[s] (TMA bytes landed), full[s] (ReLU done), sempty[s] (MMAs that read stage s complete),
//            tfull[b] (batch b accumulated), tempty[b] (batch b drained; one arrival per epilogue warp)
constexpr int PIPE_EPI_WARPS = 16, PIPE_THREADS = (PIPE_EPI_WARPS + 6) * 32, PIPE_MAX_STAGES = 3, PIPE_TBUF = 4;
struct PipeArgs { ConvTcArgs c; int nstages; uint32_t stage_bytes, magic_R, magic_Wp; };      // magic_x = ceil(2^32 / x): q / x = umulhi(q, magic_x) for the q that occur

// 32-byte global load (sm_100): one thread fetches its whole 16-channel slice of a pixel in one instruction
__device__ __forceinline__ void ldg256(const void* p, uint4& a, uint4& b) {
  asm volatile("ld.global.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n"
               : "=r"(a.x), "=r"(a.y), "=r"(a.z), "=r"(a.w), "=r"(b.x), "=r"(b.y), "=r"(b.z), "=r"(b.w) : "l"(p));
}

template <int COUT, int MODE>
__device__ __forceinline__ void load_aux(const ConvTcArgs& a, size_t o, bool valid, uint4 (&x0)[2], uint4 (&x1)[2]) {
  x0[0] = x0[1] = x1[0] = x1[1] = make_uint4(0, 0, 0, 0);
  if (!valid) return;
  if (MODE == 0) {      // (measured: the 32-byte form helps the two-operand dgrad epilogue and hurts the forward one)
    if (a.aux0) { x0[0] = *reinterpret_cast<const uint4*>(a.aux0 + o); x0[1] = *reinterpret_cast<const uint4*>(a.aux0 + o + 8); }
  } else {
    if (a.aux0) ldg256(a.aux0 + o, x0[0], x0[1]);
    if (a.aux1) ldg256(a.aux1 + o, x1[0], x1[1]);
  }
}

template <int COUT, int MODE>
__device__ __forceinline__ void finish_chunk(const ConvTcArgs& a, const float* bias_s, float (&v)[16], size_t o, int c0, const uint4 (&x0)[2], const uint4 (&x1)[2]) {
  const bf16* h0 = reinterpret_cast<const bf16*>(&x0[0]); const bf16* h1 = reinterpret_cast<const bf16*>(&x1[0]);
  if (MODE == 0) {
#pragma unroll
    for (int i = 0; i < 16; i += 4) { const float4 b4 = *reinterpret_cast<const float4*>(bias_s + c0 + i); v[i] += b4.x; v[i + 1] += b4.y; v[i + 2] += b4.z; v[i + 3] += b4.w; }
    if (a.aux0) {
#pragma unroll
      for (int i = 0; i < 16; ++i) v[i] += __bfloat162float(h0[i]);
    }
    if (a.relu_out) {
#pragma unroll
      for (int i = 0; i < 16; ++i) v[i] = fmaxf(v[i], 0.f);
    }
  } else {
    if (a.aux0) {
#pragma unroll
      for (int i = 0; i < 16; ++i) if (!(__bfloat162float(h0[i]) > 0.f)) v[i] = 0.f;
    }
    if (a.aux1) {
#pragma unroll
      for (int i = 0; i < 16; ++i) v[i] += __bfloat162float(h1[i]);
    }
  }
  uint4 o0, o1;
  __nv_bfloat162* p0 = reinterpret_cast<__nv_bfloat162*>(&o0); __nv_bfloat162* p1 = reinterpret_cast<__nv_bfloat162*>(&o1);
#pragma unroll
  for (int i = 0; i < 4; ++i) { p0[i] = __floats2bfloat162_rn(v[2 * i], v[2 * i + 1]); p1[i] = __floats2bfloat162_rn(v[8 + 2 * i], v[8 + 2 * i + 1]); }
  *reinterpret_cast<uint4*>(a.out + o) = o0;      // two 16-byte stores: measured faster than one 32-byte store here
  *reinterpret_cast<uint4*>(a.out + o + 8) = o1;
}

template <int CIN, int COUT, int MODE>
__global__ void __launch_bounds__(PIPE_THREADS) conv3x3_tc_pipe_kernel(const PipeArgs pa, const __grid_constant__ CUtensorMap tmap) {
  extern __shared__ __align__(128) uint8_t smem[];
  const ConvTcArgs& a = pa.c;
  constexpr int NCH = CIN / 8, KSTEPS = CIN / 16, TB = 128 / COUT, CPT = COUT / 16;      // tiles per batch; 16-column chunks per tile
  constexpr uint32_t W_BYTES = 9u * CIN * COUT * 2u;
  constexpr int NBAR = 3 * PIPE_MAX_STAGES + 2 * PIPE_TBUF;
  __shared__ __align__(8) uint64_t bars[NBAR];
  __shared__ uint32_t tmem_base_smem;
  __shared__ __align__(16) float bias_s[64];
  const int tid = threadIdx.x, warp = tid >> 5, NS = pa.nstages;
  const int Wp = a.W + 2, R = (a.RB + 2) * Wp;
  // stages hold whole pixels, one row of PITCH = 2*CIN bytes per position, in the 32B/64B/128B swizzle pattern the TMA writes and
  // the A descriptor names; the pattern is a function of the absolute shared-memory address (stages are 1024-byte aligned), so a
  // descriptor may start at any position: a tap is still a constant shift of the start address
  constexpr uint32_t PITCH = 2u * CIN, SWZ = CIN == 16 ? 6u : (CIN == 32 ? 4u : 2u);
  uint8_t* w_smem = smem;
  uint8_t* in_smem = smem + W_BYTES; in_smem += (1024u - (smem_u32(in_smem) & 1023u)) & 1023u;
  const uint32_t bar0 = smem_u32(&bars[0]);
  auto RAW = [&](int s) { return bar0 + 8u * (uint32_t)s; };
  auto FULL = [&](int s) { return bar0 + 8u * (uint32_t)(PIPE_MAX_STAGES + s); };
  auto SEMPTY = [&](int s) { return bar0 + 8u * (uint32_t)(2 * PIPE_MAX_STAGES + s); };
  auto TFULL = [&](int b) { return bar0 + 8u * (uint32_t)(3 * PIPE_MAX_STAGES + b); };
  auto TEMPTY = [&](int b) { return bar0 + 8u * (uint32_t)(3 * PIPE_MAX_STAGES + PIPE_TBUF + b); };
  if (tid == 0) {
    for (int i = 0; i < 3 * PIPE_MAX_STAGES + PIPE_TBUF; ++i) mbar_init(bar0 + 8u * i, 1);
    for (int b = 0; b < PIPE_TBUF; ++b) mbar_init(TEMPTY(b), PIPE_EPI_WARPS);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    tma::prefetch_map(&tmap);
  }
  if (warp == PIPE_EPI_WARPS + 1) tmem_alloc(smem_u32(&tmem_base_smem), 512);
  for (uint32_t i = tid; i < pa.stage_bytes * (uint32_t)NS / 16; i += PIPE_THREADS) reinterpret_cast<uint4*>(in_smem)[i] = make_uint4(0, 0, 0, 0);
  pdl_wait(); pdl_trigger();      // everything above is private to the CTA; everything below reads what earlier kernels wrote
  if (MODE == 0 && tid < COUT) bias_s[tid] = a.bias[tid];
  for (uint32_t i = tid; i < W_BYTES / 16; i += PIPE_THREADS) reinterpret_cast<uint4*>(w_smem)[i] = reinterpret_cast<const uint4*>(a.w)[i];
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_smem;
  const int nitems = ((a.F + a.G - 1) / a.G) * a.nbands;
  const int my_items = ((int)blockIdx.x < nitems) ? (nitems - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;

  if (warp < PIPE_EPI_WARPS) {
    // ================= epilogue =================
    constexpr int NWG = PIPE_EPI_WARPS / 4;
    const int wg = warp >> 2, lane_row = tid & 127;
    const uint32_t lane_addr = (uint32_t)((warp & 3) * 32) << 16;
    uint32_t bc = 0;      // running batch counter (same sequence as the MMA issuer)
    for (int it = 0; it < my_items; ++it) {
      const int item = blockIdx.x + it * gridDim.x;
      const int fg = item / a.nbands, yb = (item - fg * a.nbands) * a.RB, f0 = fg * a.G, nf = min(a.G, a.F - f0);
      const int ntiles = ((nf - 1) * R + a.RB * Wp + 127) / 128;
      for (int t0 = 0; t0 < ntiles; t0 += TB, ++bc) {
        const int nt = min(TB, ntiles - t0), b = (int)(bc % PIPE_TBUF);
        const int npairs = (nt > wg ? (nt - wg - 1) / NWG + 1 : 0) * CPT;      // (tile, 16-column chunk) pairs of this warpgroup
        auto locate = [&](int u, size_t& o, bool& valid, uint32_t& col) {
          const int s = wg + NWG * (u / CPT), c0 = (u % CPT) * 16;
          const int q = (t0 + s) * 128 + lane_row, j = (int)__umulhi((uint32_t)q, pa.magic_R), rem = q - j * R;
          const int yl = (int)__umulhi((uint32_t)rem, pa.magic_Wp), x = rem - yl * Wp, y = yb + yl;
          valid = j < nf && yl < a.RB && y < a.H && x < a.W;
          o = (((size_t)(f0 + j) * a.H + y) * a.W + x) * COUT + c0;
          col = (uint32_t)(b * 128 + s * COUT + c0);
        };
        size_t o = 0; bool valid = false; uint32_t col = 0; uint4 x0[2], x1[2];
        if (npairs > 0) { locate(0, o, valid, col); load_aux<COUT, MODE>(a, o, valid, x0, x1); }      // before the wait: latency hidden
        if (!mbar_wait(TFULL(b), (bc / PIPE_TBUF) & 1u)) { if (a.error_flag) *a.error_flag = 1; }
        tc_fence_after();
        for (int u = 0; u < npairs; ++u) {
          size_t o_n = 0; bool valid_n = false; uint32_t col_n = 0; uint4 n0[2], n1[2];
          if (u + 1 < npairs) { locate(u + 1, o_n, valid_n, col_n); load_aux<COUT, MODE>(a, o_n, valid_n, n0, n1); }
          float v[16];
          tmem_ld16(tmem_base + lane_addr + col, v);
          if (valid) finish_chunk<COUT, MODE>(a, bias_s, v, o, (int)(col % COUT), x0, x1);
          o = o_n; valid = valid_n; col = col_n; x0[0] = n0[0]; x0[1] = n0[1]; x1[0] = n1[0]; x1[1] = n1[1];
        }
        tc_fence_before();
        __syncwarp();
        if ((tid & 31) == 0) asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}\n" :: "r"(TEMPTY(b)) : "memory");
      }
    }
  } else if (warp == PIPE_EPI_WARPS) {
    // ================= TMA producer =================
    const uint32_t bytes = (uint32_t)(a.G * R) * 16u * NCH;
    for (int it = 0; it < my_items; ++it) {
      const int item = blockIdx.x + it * gridDim.x, s = it % NS, use = it / NS;
      const int fg = item / a.nbands, yb = (item - fg * a.nbands) * a.RB, f0 = fg * a.G;
      if (use > 0 && !mbar_wait(SEMPTY(s), (uint32_t)((use - 1) & 1))) { if (a.error_flag) *a.error_flag = 6; }
      if (elect_one()) {
        const uint32_t dst = smem_u32(in_smem) + (uint32_t)s * pa.stage_bytes;
        tma::arrive_expect_tx(RAW(s), bytes);
        tma::load_4d(dst, &tmap, 0, -1, yb - 1, f0, RAW(s));
      }
      __syncwarp();
    }
  } else if (warp == PIPE_EPI_WARPS + 1) {
    // ================= MMA issuer =================
    const uint32_t idesc = make_idesc(128, COUT, 0, 0);
    const uint32_t d_hi = 8u | (1u << 14);                                                                    // B: SBO = 128 B, version bit 46
    const uint32_t a_hi = ((8u * PITCH) >> 4) | (1u << 14) | (SWZ << 29);                                     // A: SBO = 8 rows, swizzle mode in bits 61-63
    const uint32_t b_lo = ((smem_u32(w_smem) >> 4) & 0x3FFFu) | ((uint32_t)COUT << 16);                       // LBO = COUT*16 B
    uint32_t bc = 0;
    for (int it = 0; it < my_items; ++it) {
      const int item = blockIdx.x + it * gridDim.x, s = it % NS, use = it / NS;
      const int fg = item / a.nbands, f0 = fg * a.G, nf = min(a.G, a.F - f0);
      const int ntiles = ((nf - 1) * R + a.RB * Wp + 127) / 128;
      if (!mbar_wait(a.relu_in ? FULL(s) : RAW(s), (uint32_t)(use & 1))) { if (a.error_flag) *a.error_flag = 2; }
      tc_fence_after();
      const uint32_t a_lo = (((smem_u32(in_smem) + (uint32_t)s * pa.stage_bytes) >> 4) & 0x3FFFu) | (1u << 16);      // LBO unused (one swizzle row holds the K slice)
      for (int t0 = 0; t0 < ntiles; t0 += TB, ++bc) {
        const int nt = min(TB, ntiles - t0), b = (int)(bc % PIPE_TBUF);
        if (bc >= PIPE_TBUF && !mbar_wait(TEMPTY(b), ((bc / PIPE_TBUF) - 1) & 1u)) { if (a.error_flag) *a.error_flag = 3; }
        tc_fence_after();
#pragma unroll 1
        for (int sT = 0; sT < nt; ++sT) {
          const uint32_t td = tmem_base + (uint32_t)(b * 128 + sT * COUT);
          uint32_t row_lo = a_lo + (uint32_t)(t0 + sT) * 128u * (PITCH >> 4);      // start of the tile, tap row di = 0
          uint32_t acc = 0;
#pragma unroll
          for (int di = 0; di < 3; ++di) {
#pragma unroll
            for (int dj = 0; dj < 3; ++dj) {
#pragma unroll
              for (int ks = 0; ks < KSTEPS; ++ks) {
                const uint64_t ad = ((uint64_t)a_hi << 32) | (uint64_t)(row_lo + (uint32_t)(dj * (PITCH >> 4) + 2 * ks));
                const uint64_t bd = ((uint64_t)d_hi << 32) | (uint64_t)(b_lo + (uint32_t)(((di * 3 + dj) * NCH + 2 * ks) * COUT));
                if (elect_one()) mma_f16(td, ad, bd, idesc, acc);
                acc = 1;
              }
            }
            row_lo += (uint32_t)Wp * (PITCH >> 4);
          }
        }
        if (elect_one()) {
          mma_commit(TFULL(b));
          if (t0 + TB >= ntiles) mma_commit(SEMPTY(s));      // last batch of the item: the stage may be refilled once these MMAs are done
        }
        __syncwarp();
      }
    }
  } else if (a.relu_in) {
    // ================= ReLU in place on a landed stage (the last four warps) =================
    const int t = tid - (PIPE_EPI_WARPS + 2) * 32, n16 = a.G * R;
    for (int it = 0; it < my_items; ++it) {
      const int s = it % NS, use = it / NS;
      if (!mbar_wait(RAW(s), (uint32_t)(use & 1))) { if (a.error_flag) *a.error_flag = 7; }
      uint4* st = reinterpret_cast<uint4*>(in_smem + (size_t)s * pa.stage_bytes);
      const __nv_bfloat162 z = __float2bfloat162_rn(0.f);
      // elementwise (the swizzle does not matter); four independent 16-byte loads in flight per thread: the pass sits on the critical path
      // between the TMA landing and the first MMA of the item (measured: 2.4 us per 62 KB stage with one load in flight, against a 4.5 us item)
      const int tot = n16 * NCH;
      for (int i0 = t; i0 < tot; i0 += 4 * 128) {
        uint4 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) if (i0 + u * 128 < tot) v[u] = st[i0 + u * 128];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          if (i0 + u * 128 >= tot) break;
          __nv_bfloat162* h = reinterpret_cast<__nv_bfloat162*>(&v[u]);
#pragma unroll
          for (int k = 0; k < 4; ++k) h[k] = __hmax2(h[k], z);
          st[i0 + u * 128] = v[u];
        }
      }
      fence_async_smem();
      asm volatile("bar.sync 2, 128;\n" ::: "memory");
      if (t == 0) asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}\n" :: "r"(FULL(s)) : "memory");
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == PIPE_EPI_WARPS + 1) tmem_dealloc(tmem_base, 512);
}

}  // namespace tc

// ---- host side ---------------------------------------------------------------------------------
bool conv_tc_supported(const Geom& g) {
  auto okc = [](int c) { return c == 16 || c == 32 || c == 64; };
  // the kernel is fed by TMA: without cuTensorMapEncodeTiled (or with CB_DISABLE_TMA=1) the layer runs on the SIMT implicit GEMM
  return g.kh == 3 && g.kw == 3 && g.s == 1 && g.p == 1 && okc(g.Cin) && okc(g.Cout) && g.H == g.Ho && g.W == g.Wo && tma::encode_fn() != nullptr;
}

// plan of the pipelined kernel: NS stages of one item (G whole frames, or one row band of one frame) in <= 200 KB with the weights
struct PipePlan { int G, npix_alloc, RB, nbands, nstages; size_t stage_bytes, smem; bool ok; };
static PipePlan pipe_plan(int F, int H, int W, int cin, int cout) {
  const int Wp = W + 2, R = (H + 2) * Wp;
  const size_t wbytes = ((size_t)9 * cin * cout * 2 + 127) & ~(size_t)127;
  const size_t avail = (size_t)200 * 1024 - wbytes - 1024;      // 1 KB: the stages start on a 1024-byte boundary
  auto alloc_pix = [&](int positions) { int n = ((positions + 127) / 128) * 128 + 2 * Wp + 2; return (n + 7) / 8 * 8; };
  auto bytes = [&](int positions) { return ((size_t)alloc_pix(positions) * cin * 2 + 1023) & ~(size_t)1023; };
  PipePlan p{1, 0, H, 1, 3, 0, 0, true};
  if (bytes(R) <= avail / 3) {
    // whole frames: the group size that minimises (items of the busiest CTA) x (tiles per item); a function of the shape only
    long best = -1;
    for (int G = 1; G <= 8 && bytes(G * R) <= avail / 3; ++G) {
      const long items = (F + G - 1) / G, per_cta = (items + 147) / 148, tiles = ((long)(G - 1) * R + (long)H * Wp + 127) / 128;
      const long cost = per_cta * (tiles * 9 + 12);      // + a fixed per-item hand-off cost, in units of one tap
      if (best < 0 || cost < best) { best = cost; p.G = G; }
    }
    p.npix_alloc = alloc_pix(p.G * R);
  } else if (bytes(R) <= avail / 2) {
    p.nstages = 2; p.npix_alloc = alloc_pix(R);
  } else {
    p.nstages = 2;
    long rows = ((long)(avail / 2) / ((long)cin * 2) - 2 * Wp - 140) / Wp - 2;
    if (rows < 2) { p.ok = false; return p; }
    p.nbands = (int)((H + rows - 1) / rows); p.RB = (H + p.nbands - 1) / p.nbands;
    p.npix_alloc = alloc_pix((p.RB + 2) * Wp);
  }
  p.stage_bytes = ((size_t)p.npix_alloc * cin * 2 + 1023) & ~(size_t)1023;
  p.smem = wbytes + 1024 + (size_t)p.nstages * p.stage_bytes;
  p.ok = p.smem <= (size_t)220 * 1024;
  return p;
}

// the staged items plus the weight image must fit one CTA's shared memory
bool conv_tc_fits(int H, int W, int cin, int cout) { return pipe_plan(148, H, W, cin, cout).ok; }

template <int CIN, int COUT, int MODE>
static int launch_pipe(const tc::PipeArgs& a, const CUtensorMap& tmap, size_t smem, int nitems, cudaStream_t st) {
  { int rc = ensure_dyn_smem((const void*)tc::conv3x3_tc_pipe_kernel<CIN, COUT, MODE>, smem); if (rc) return rc; }
  CB_CUDA(launch_pdl(tc::conv3x3_tc_pipe_kernel<CIN, COUT, MODE>, dim3(std::min(nitems, 148)), dim3(tc::PIPE_THREADS), smem, st, a, tmap));
  return CB_OK;
}

template <int MODE>
static int dispatch_pipe(int cin, int cout, const tc::PipeArgs& a, const CUtensorMap& tmap, size_t smem, int nitems, cudaStream_t st) {
#define CB_TC_CASE(ci, co) if (cin == ci && cout == co) return launch_pipe<ci, co, MODE>(a, tmap, smem, nitems, st);
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
  CUtensorMap tmap; memset(&tmap, 0, sizeof tmap);
  {      // pipelined, TMA-fed kernel
    const PipePlan q = pipe_plan(F, H, W, cin, cout);
    if (q.ok && W + 2 <= 256 && q.RB + 2 <= 256 && tma::make_nhwc_map(&tmap, in, F, H, W, cin, W + 2, q.RB + 2, q.G, cin, true)) {
      tc::PipeArgs pa{{in, w, bias, aux0, aux1, out, F, H, W, q.G, q.npix_alloc, relu_in ? 1 : 0, 1, relu_out ? 1 : 0, q.RB, q.nbands, error_flag},
                      q.nstages, (uint32_t)q.stage_bytes, (uint32_t)((0x100000000ull + (uint64_t)((q.RB + 2) * (W + 2)) - 1) / (uint64_t)((q.RB + 2) * (W + 2))),
                      (uint32_t)((0x100000000ull + (uint64_t)(W + 2) - 1) / (uint64_t)(W + 2))};
      const int nitems = ((F + q.G - 1) / q.G) * q.nbands;
      return mode == 0 ? dispatch_pipe<0>(cin, cout, pa, tmap, q.smem, nitems, st) : dispatch_pipe<1>(cin, cout, pa, tmap, q.smem, nitems, st);
    }
  }
  set_error("conv_tc: no plan for this shape, or the driver refused the tensor map");
  return CB_ECUDA;
}

}  // namespace cb
