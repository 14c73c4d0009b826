// Network side of the hot path: weight packing, forward and backward
// (a9-a10) over the layer program built in api.cu.  Plain SIMT path; tcgen05 kernels live in
// conv_tc.cu and are dispatched from here when the shape qualifies.
#include "gemm_simt.cuh"
#include "pool.cuh"

#include <type_traits>

namespace cb {

// ---- weight packing: canonical fp32 [Cout,Cin,kh,kw] -> Wf [(di,dj,c)][n], Wd [(di,dj,n)][c], bias fp32 [n]
template <typename AT>
__global__ void pack_kernel(const float* __restrict__ params, Geom g, ParamMap pm, AT* wf, AT* wd, float* bias) {
  int K = g.kh * g.kw * g.Cin;
  size_t total = (size_t)K * g.Cout;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    int n = (int)(i % g.Cout); int k = (int)(i / g.Cout);
    int c = k % g.Cin; int q = k / g.Cin; int dj = q % g.kw, di = q / g.kw;
    float v = params[pm.w(n, c, di, dj, g)];
    stv(wf, i, v);
    stv(wd, ((size_t)(di * g.kw + dj) * g.Cout + n) * g.Cin + c, v);
    if (k == 0) bias[n] = params[pm.b(n)];
  }
}

// tcgen05 B operands (conv_tc.cu): forward [tap][Cin/8][Cout][8]; dgrad [tap'][Cout/8][Cin][8] with flipped taps
__global__ void pack_tc_kernel(const float* __restrict__ params, Geom g, ParamMap pm, bf16* wtf, bf16* wtd) {
  size_t total = (size_t)9 * g.Cin * g.Cout;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    int n = (int)(i % g.Cout); size_t q = i / g.Cout; int c = (int)(q % g.Cin); int tap = (int)(q / g.Cin);
    int di = tap / 3, dj = tap % 3;
    bf16 v = __float2bfloat16_rn(params[pm.w(n, c, di, dj, g)]);
    wtf[(((size_t)tap * (g.Cin / 8) + c / 8) * g.Cout + n) * 8 + c % 8] = v;
    int tapd = (2 - di) * 3 + (2 - dj);
    wtd[(((size_t)tapd * (g.Cout / 8) + n / 8) * g.Cin + c) * 8 + n % 8] = v;
  }
}

// all layers in ONE launch: blockIdx.y = layer, blocks of a layer stride over its weights.  Per weight element:
// Wf, Wd (SIMT operands), bias, and for the tensor-core layers the B-operand images of conv_tc.cu / conv0_tc.cu.
template <typename AT>
__global__ void pack_all_kernel(const float* __restrict__ params, const PackDesc* __restrict__ tab, AT* wf_all, AT* wd_all, float* bias_all,
                                bf16* wtf_all, bf16* wtd_all, bf16* w0img) {
  const PackDesc d = tab[blockIdx.y];
  const Geom g = d.g;
  const int K = g.kh * g.kw * g.Cin;
  const size_t total = (size_t)K * g.Cout;
  AT* wf = wf_all + d.wf_off; AT* wd = wd_all + d.wf_off; float* bias = bias_all + d.bias_off;
  // four elements per pass: their (strided) fp32 reads are issued together, then the stores follow
  const uint32_t stride = gridDim.x * blockDim.x, tot = (uint32_t)total;
  for (uint32_t i0 = blockIdx.x * blockDim.x + threadIdx.x; i0 < tot; i0 += 4 * stride) {
    float v4[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const uint32_t i = i0 + u * stride;
      v4[u] = 0.f;
      if (i < tot) {
        int n = (int)(i % (uint32_t)g.Cout); int k = (int)(i / (uint32_t)g.Cout);
        int c = k % g.Cin; int q = k / g.Cin; int dj = q % g.kw, di = q / g.kw;
        v4[u] = __ldg(params + d.pm.w(n, c, di, dj, g));
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const uint32_t i = i0 + u * stride;
      if (i >= tot) break;
      const float v = v4[u];
      int n = (int)(i % (uint32_t)g.Cout); int k = (int)(i / (uint32_t)g.Cout);
      int c = k % g.Cin; int q = k / g.Cin; int dj = q % g.kw, di = q / g.kw;
      stv(wf, i, v);
      stv(wd, ((size_t)(di * g.kw + dj) * g.Cout + n) * g.Cin + c, v);
      if (k == 0) bias[n] = params[d.pm.b(n)];
      if (d.tc) {
        const int tap = di * 3 + dj, tapd = (2 - di) * 3 + (2 - dj);
        const bf16 h = __float2bfloat16_rn(v);
        (wtf_all + d.wf_off)[(((size_t)tap * (g.Cin / 8) + c / 8) * g.Cout + n) * 8 + c % 8] = h;
        (wtd_all + d.wf_off)[(((size_t)tapd * (g.Cout / 8) + n / 8) * g.Cin + c) * 8 + n % 8] = h;
      }
    }
  }
  if (d.dense) {      // dense_tc.cu forward B operand [N][K] (k = (y, x, c)): thread = (n, 8-channel group, pixel), pixel fastest, so that the canonical
    // [n][c][y][x] reads are contiguous across threads; each thread writes one 16-byte vector
    const uint32_t npix = (uint32_t)(g.kh * g.kw), c8n = (uint32_t)g.Cin / 8, totd = (uint32_t)g.Cout * c8n * npix;
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < totd; i += stride) {
      const uint32_t pix = i % npix, q = i / npix, c8 = q % c8n, n = q / c8n;
      const int di = (int)(pix / (uint32_t)g.kw), dj = (int)(pix % (uint32_t)g.kw);
      float f[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) f[j] = __ldg(params + d.pm.w((int)n, (int)(c8 * 8 + j), di, dj, g));
      __nv_bfloat162 o[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) o[j] = __floats2bfloat162_rn(f[2 * j], f[2 * j + 1]);
      *reinterpret_cast<uint4*>(wtf_all + d.wf_off + (size_t)n * K + (size_t)pix * g.Cin + c8 * 8) = *reinterpret_cast<const uint4*>(o);
    }
  }
  if (d.conv0) {      // forward B image [slot = 2*di + h][chunk][o][8]: chunks (di, 2h), (di, 2h+1); channels >= Cin and dj = 3 are zero
    const int tot0 = 6 * 2 * g.Cout * 8;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < tot0; i += gridDim.x * blockDim.x) {
      int c = i & 7, o = (i >> 3) % g.Cout, chunk = ((i >> 3) / g.Cout) & 1, slot = (i >> 3) / g.Cout / 2;
      int di = slot >> 1, dj = (slot & 1) * 2 + chunk;
      float v = (c < g.Cin && dj < 3) ? params[d.pm.w(o, c, di, dj, g)] : 0.f;
      w0img[i] = __float2bfloat16_rn(v);
    }
    // pixel-pair image (conv0_fwd_ws_kernel): [di][chunk][n = e Cout + o][8]; K index kk = 8 chunk + col = 4 j + c (input position j of the four a
    // pair reads, channel c); pixel e of the pair sees position j as tap dj = j - e
    bf16* img2 = w0img + tot0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < tot0; i += gridDim.x * blockDim.x) {
      const int col = i & 7, n = (i >> 3) % (2 * g.Cout), chunk = ((i >> 3) / (2 * g.Cout)) & 1, di = (i >> 3) / (2 * g.Cout) / 2;
      const int kk = 8 * chunk + col, j = kk >> 2, c = kk & 3, e = n / g.Cout, o = n - e * g.Cout, dj = j - e;
      const float v = (c < g.Cin && dj >= 0 && dj < 3) ? params[d.pm.w(o, c, di, dj, g)] : 0.f;
      img2[i] = __float2bfloat16_rn(v);
    }
  }
}

template <typename AT>
static int pack_all(cb_net* net, Workspace& ws, const float* params, cudaStream_t st) {
  ProfScope ps(K_PACK, st, 1, 0.0, (double)net->P * (4 + 2 * sizeof(AT)));
  dim3 grid(296, (unsigned)net->layers.size());      // the fc layer holds 90 % of the elements: enough CTAs to cover its strided reads
  pack_all_kernel<AT><<<grid, 256, 0, st>>>(params, ws.packtab, (AT*)ws.wf, (AT*)ws.wd, ws.bias, ws.wtc_f, ws.wtc_d, ws.w0img);
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

int pack_weights(cb_net* net, int prec, const float* params, cudaStream_t st) {
  Workspace& ws = net->ws[prec];
  ws.packed = true;
  return prec == CB_PREC_FP32_REF ? pack_all<float>(net, ws, params, st) : pack_all<bf16>(net, ws, params, st);
}

// ---- max-pool 3x3 stride 2, XLA-SAME padding (A10), NHWC ------------------------------------
__host__ __device__ inline int pool_out(int h) { return (h + 1) / 2; }
__host__ __device__ inline int pool_pad_lo(int h) { int o = pool_out(h); int tot = (o - 1) * 2 + 3 - h; if (tot < 0) tot = 0; return tot / 2; }

template <typename AT>
__global__ void pool_fwd_kernel(const AT* __restrict__ x, AT* __restrict__ y, int F, int C, int H, int W) {
  int Ho = pool_out(H), Wo = pool_out(W), ph = pool_pad_lo(H), pw = pool_pad_lo(W);
  size_t total = (size_t)F * Ho * Wo * C;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    int c = (int)(i % C); size_t q = i / C; int ox = (int)(q % Wo); q /= Wo; int oy = (int)(q % Ho); size_t f = q / Ho;
    float best = -INFINITY;
    for (int di = 0; di < 3; ++di) {
      int iy = oy * 2 + di - ph; if ((unsigned)iy >= (unsigned)H) continue;
      for (int dj = 0; dj < 3; ++dj) {
        int ix = ox * 2 + dj - pw; if ((unsigned)ix >= (unsigned)W) continue;
        float v = ldv(x, ((f * H + iy) * W + ix) * C + c);
        if (v > best) best = v;
      }
    }
    stv(y, i, best);
  }
}

// gather form of the adjoint: input pixel (iy,ix) receives dy of every window whose FIRST maximum
// in row-major window order (A11) is this pixel.  No atomics.
template <typename AT>
__global__ void pool_bwd_kernel(const AT* __restrict__ x, const AT* __restrict__ dy, AT* __restrict__ dx, int F, int C, int H, int W) {
  int Ho = pool_out(H), Wo = pool_out(W), ph = pool_pad_lo(H), pw = pool_pad_lo(W);
  size_t total = (size_t)F * H * W * C;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    int c = (int)(i % C); size_t q = i / C; int ix = (int)(q % W); q /= W; int iy = (int)(q % H); size_t f = q / H;
    float g = 0.f;
    // windows containing (iy,ix): oy*2 - ph <= iy <= oy*2 - ph + 2
    int oy_lo = (iy + ph - 2 + 1) / 2; if (iy + ph - 2 < 0) oy_lo = 0;
    int ox_lo = (ix + pw - 2 + 1) / 2; if (ix + pw - 2 < 0) ox_lo = 0;
    int oy_hi = min((iy + ph) / 2, Ho - 1), ox_hi = min((ix + pw) / 2, Wo - 1);
    for (int oy = oy_lo; oy <= oy_hi; ++oy)
      for (int ox = ox_lo; ox <= ox_hi; ++ox) {
        float best = -INFINITY; int by = -1, bx = -1;
        for (int di = 0; di < 3; ++di) {
          int yy = oy * 2 + di - ph; if ((unsigned)yy >= (unsigned)H) continue;
          for (int dj = 0; dj < 3; ++dj) {
            int xx = ox * 2 + dj - pw; if ((unsigned)xx >= (unsigned)W) continue;
            float v = ldv(x, ((f * H + yy) * W + xx) * C + c);
            if (v > best) { best = v; by = yy; bx = xx; }
          }
        }
        if (by == iy && bx == ix) g += ldv(dy, ((f * Ho + oy) * Wo + ox) * C + c);
      }
    stv(dx, i, g);
  }
}

// 8-channel (16-byte) vectorised variants for bf16 maps with C % 8 == 0: one thread per (pixel, chunk)
__device__ __forceinline__ void bf8_to_f(const uint4& u, float* f) {
  const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&u);
#pragma unroll
  for (int i = 0; i < 4; ++i) { float2 t = __bfloat1622float2(h[i]); f[2 * i] = t.x; f[2 * i + 1] = t.y; }
}
__device__ __forceinline__ uint4 f_to_bf8(const float* f) {
  uint4 u; __nv_bfloat162* h = reinterpret_cast<__nv_bfloat162*>(&u);
#pragma unroll
  for (int i = 0; i < 4; ++i) h[i] = __floats2bfloat162_rn(f[2 * i], f[2 * i + 1]);
  return u;
}
// IT = index type of the element counter: uint32_t whenever F*Ho*Wo*C/8 < 2^32 (64-bit divisions cost more than the window maximum)
template <typename IT>
__global__ void pool_fwd_v8_kernel(const bf16* __restrict__ x, bf16* __restrict__ y, uint8_t* __restrict__ arg, int F, int C, int H, int W) {
  int Ho = pool_out(H), Wo = pool_out(W), ph = pool_pad_lo(H), pw = pool_pad_lo(W), C8 = C / 8;
  const IT total = (IT)F * (IT)Ho * (IT)Wo * (IT)C8;
  for (IT i = blockIdx.x * (IT)blockDim.x + threadIdx.x; i < total; i += (IT)gridDim.x * blockDim.x) {
    int c8 = (int)(i % (IT)C8); IT q = i / (IT)C8; int ox = (int)(q % (IT)Wo); q /= (IT)Wo; int oy = (int)(q % (IT)Ho); size_t f = (size_t)(q / (IT)Ho);
    uint4 v[9]; uint32_t valid = 0;
#pragma unroll
    for (int di = 0; di < 3; ++di) {
      const int iy = oy * 2 + di - ph;
#pragma unroll
      for (int dj = 0; dj < 3; ++dj) {
        const int ix = ox * 2 + dj - pw;
        if ((unsigned)iy < (unsigned)H && (unsigned)ix < (unsigned)W) {
          v[di * 3 + dj] = *reinterpret_cast<const uint4*>(x + ((f * H + iy) * W + ix) * C + c8 * 8);
          valid |= 1u << (di * 3 + dj);
        }
      }
    }
    uint4 best; uint2 pk;
    pool::window_max(v, valid, best, pk);      // packed bf16 max; first maximum in window order (A11)
    *reinterpret_cast<uint4*>(y + (size_t)i * 8) = best;
    *reinterpret_cast<uint2*>(arg + (size_t)i * 8) = pk;
  }
}
// Max-pool adjoint, scatter form: one CTA builds a band of `RB` input rows of one frame in shared memory.  Every
// pooled element of the rows that reach into the band adds its gradient to the pixel its stored arg-max names.
// Windows whose (oy, ox) parities agree are disjoint, so the four parity classes run as four barrier-separated
// phases of plain read-modify-writes (no atomics, fixed order: bitwise reproducible); a pixel elected by several
// windows is rounded to bf16 after each addition.  The finished band leaves as one linear copy.
__global__ void __launch_bounds__(256) pool_bwd_scatter_kernel(const uint8_t* __restrict__ arg, const bf16* __restrict__ dy, bf16* __restrict__ dx,
                                                               int F, int C, int H, int W, int RB, int nbands) {
  asm volatile("griddepcontrol.wait;\n" ::: "memory");      // launched through launch_pdl: resident before its predecessor has drained
  asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory");
  extern __shared__ __align__(16) uint8_t tile[];
  const int Ho = pool_out(H), Wo = pool_out(W), ph = pool_pad_lo(H), pw = pool_pad_lo(W), C8 = C / 8, tid = threadIdx.x;
  for (int item = blockIdx.x; item < F * nbands; item += gridDim.x) {
    const int f = item / nbands, yb = (item - f * nbands) * RB, rows = min(RB, H - yb);
    const int n16 = rows * W * C8;
    int lo = yb + ph - 2; lo = lo <= 0 ? 0 : (lo + 1) / 2;
    const int hi = min((yb + rows - 1 + ph) / 2, Ho - 1);
    // this thread's first element of each phase is fetched before the tile is touched
    uint2 pk[4]; uint4 dv[4]; int py[4], px[4], pc[4]; bool ok[4];
#pragma unroll
    for (int p = 0; p < 4; ++p) {
      const int pa = p >> 1, pb = p & 1, first = lo + (((lo & 1) != pa) ? 1 : 0);
      const int noy = hi >= first ? (hi - first) / 2 + 1 : 0, nox = (Wo - pb + 1) / 2;
      ok[p] = tid < noy * nox * C8;
      if (ok[p]) {
        pc[p] = tid % C8; const int r = tid / C8; px[p] = pb + 2 * (r % nox); py[p] = first + 2 * (r / nox);
        const size_t o = (((size_t)f * Ho + py[p]) * Wo + px[p]) * C + pc[p] * 8;
        pk[p] = pool::ldg_early_v2(arg + o); dv[p] = pool::ldg_early_v4(dy + o);      // issued here, ahead of the zero fill and the barriers
      }
    }
    for (int i = tid; i < n16; i += 256) reinterpret_cast<uint4*>(tile)[i] = make_uint4(0, 0, 0, 0);
#pragma unroll
    for (int p = 0; p < 4; ++p) {
      __syncthreads();
      const int pa = p >> 1, pb = p & 1, first = lo + (((lo & 1) != pa) ? 1 : 0);
      const int noy = hi >= first ? (hi - first) / 2 + 1 : 0, nox = (Wo - pb + 1) / 2, n = noy * nox * C8;
      for (int i = tid; i < n; i += 256) {
        int oy, ox, c8; uint2 k2; uint4 d4;
        if (i == tid && ok[p]) { oy = py[p]; ox = px[p]; c8 = pc[p]; k2 = pk[p]; d4 = dv[p]; }
        else {
          c8 = i % C8; const int r = i / C8; ox = pb + 2 * (r % nox); oy = first + 2 * (r / nox);
          const size_t o = (((size_t)f * Ho + oy) * Wo + ox) * C + c8 * 8;
          k2 = *reinterpret_cast<const uint2*>(arg + o); d4 = *reinterpret_cast<const uint4*>(dy + o);
        }
        const int y0 = oy * 2 - ph - yb, x0 = ox * 2 - pw;
        const uint16_t* h = reinterpret_cast<const uint16_t*>(&d4);
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const uint32_t a = ((k < 4 ? k2.x : k2.y) >> (8 * (k & 3))) & 255u;
          const int wy = (int)((a * 11u) >> 5), wx = (int)a - 3 * wy, yl = y0 + wy;
          if ((unsigned)yl < (unsigned)rows)
            pool::add_bf16(reinterpret_cast<uint16_t*>(tile) + ((size_t)(yl * W + x0 + wx) * C + c8 * 8 + k), h[k]);
        }
      }
    }
    __syncthreads();
    uint4* out = reinterpret_cast<uint4*>(dx + ((size_t)f * H + yb) * W * C);
    for (int i = tid; i < n16; i += 256) out[i] = reinterpret_cast<const uint4*>(tile)[i];
    __syncthreads();
  }
}

// ---- wgrad second pass: sum split-K partials in split order, scale, scatter to canonical grad ----
__global__ void wgrad_reduce_kernel(const float* __restrict__ partial, int splits, Geom g, ParamMap pm, float in_scale, float* __restrict__ grad) {
  int Kw = g.kh * g.kw * g.Cin, M = Kw + 1, N = g.Cout;
  size_t total = (size_t)M * N;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    float s = 0.f;
    int z = 0;
    for (; z + 16 <= splits; z += 16) {      // 16 loads in flight, then the additions in z order
      float v[16];
#pragma unroll
      for (int k = 0; k < 16; ++k) v[k] = __ldg(partial + (size_t)(z + k) * total + i);
#pragma unroll
      for (int k = 0; k < 16; ++k) s += v[k];
    }
    for (; z < splits; ++z) s += partial[(size_t)z * total + i];
    int n = (int)(i % N), m = (int)(i / N);
    if (m == Kw) { grad[pm.b(n)] = s; continue; }
    int c = m % g.Cin; int q = m / g.Cin; int dj = q % g.kw, di = q / g.kw;
    grad[pm.w(n, c, di, dj, g)] = s * in_scale;
  }
}

// ---- weight gradient of the two heads (a [fc x (A+1)] matrix): CTA z sums a fixed chunk of frames, thread k owns hidden unit k ----
// partial layout = [z][fc + 1][N] (row fc = bias gradient), the layout wgrad_reduce_kernel sums in z order.
constexpr int HEAD_WGRAD_SPLITS = 148;      // a constant, not the device's SM count: the summation order is a function of the shape only (A16)
template <typename AT>
__global__ void __launch_bounds__(256) heads_wgrad_kernel(const AT* __restrict__ hid, const AT* __restrict__ dy, float* __restrict__ partial, int F, int fc, int N, int chunk) {
  __shared__ float dys[64 * 32];
  const int f0 = blockIdx.x * chunk, f1 = min(F, f0 + chunk);
  float* out = partial + (size_t)blockIdx.x * (fc + 1) * N;
  for (int k0 = 0; k0 < fc + 1; k0 += 256) {
    const int k = k0 + threadIdx.x;
    float acc[32];
#pragma unroll
    for (int n = 0; n < 32; ++n) acc[n] = 0.f;
    for (int fb = f0; fb < f1; fb += 64) {
      const int nf = min(64, f1 - fb);
      __syncthreads();
      for (int i = threadIdx.x; i < nf * N; i += 256) dys[(i / N) * 32 + i % N] = (float)dy[(size_t)fb * N + i];
      __syncthreads();
      if (k <= fc)
        for (int j = 0; j < nf; ++j) {
          const float h = k < fc ? fmaxf((float)hid[(size_t)(fb + j) * fc + k], 0.f) : 1.f;
#pragma unroll
          for (int n = 0; n < 32; ++n) if (n < N) acc[n] = fmaf(h, dys[j * 32 + n], acc[n]);
        }
    }
    if (k <= fc) {
#pragma unroll
      for (int n = 0; n < 32; ++n) if (n < N) out[(size_t)k * N + n] = acc[n];
    }
  }
}

// split-K policy: a function of the problem shape only (never of the device), so the summation
// order -- and with it every bit of the gradient -- is fixed (A16).
static inline void wgrad_split(long long K, int* splits, int* kchunk, long long tiles_mn = 1 << 20) {
  const int target = tiles_mn >= 64 ? 4096 : 256;      // few output tiles: split deeper so that the grid fills the GPU
  long long s = (K + target - 1) / target; if (s < 1) s = 1; if (s > 2048) s = 2048;
  long long ch = (K + s - 1) / s; ch = (ch + 15) / 16 * 16;
  *splits = (int)((K + ch - 1) / ch); *kchunk = (int)ch;
}

size_t wgrad_partial_elems(const Geom& g, long long frames) {
  int s, ch; wgrad_split(frames * g.Ho * g.Wo, &s, &ch, (long long)((g.kh * g.kw * g.Cin + 1 + 127) / 128) * ((g.Cout + 63) / 64));
  if (g.kh == 1 && g.kw == 1 && g.H == 1 && g.W == 1 && g.Cout <= 32) s = std::max(s, HEAD_WGRAD_SPLITS);      // heads_wgrad_kernel
  return (size_t)s * (g.kh * g.kw * g.Cin + 1) * g.Cout;
}

static inline int grid_for(size_t total) { return (int)std::min<size_t>((total + 255) / 256, (size_t)148 * 16); }

template <typename AT>
static int forward_t(cb_net* net, Workspace& ws, const uint8_t* obs, const int32_t* frame_idx, int F, cudaStream_t st, bool skip_heads,
                     const int32_t* taken, int n_taken, float* logp_taken) {
  bool pool_fused = false;      // the first layer's kernel also produced the pooled map: skip the following POOL op
  for (size_t oi = 0; oi < net->fwd.size(); ++oi) {
    const Op& op = net->fwd[oi];
    if (skip_heads && op.kind == OP_CONV && net->layers[op.layer].f32_out) continue;
    if (op.kind == OP_POOL && pool_fused) { pool_fused = false; continue; }
    if (op.kind == OP_POOL) {
      size_t total = (size_t)F * pool_out(op.H) * pool_out(op.W) * op.C;
      ProfScope ps(K_POOL_FWD, st, 1, 0.0, (double)sizeof(AT) * (total + (double)F * op.H * op.W * op.C));
      if (std::is_same<AT, bf16>::value && op.C % 8 == 0)
      {
        // grid-stride counter + one stride must stay below 2^32 for the 32-bit form
        if (total / 8 + (size_t)grid_for(total / 8) * 256 < 0xFFFFFFFFull)
          pool_fwd_v8_kernel<uint32_t><<<grid_for(total / 8), 256, 0, st>>>((const bf16*)ws.act[op.in_t], (bf16*)ws.act[op.out_t], (uint8_t*)ws.act[op.mask_t], F, op.C, op.H, op.W);
        else
          pool_fwd_v8_kernel<size_t><<<grid_for(total / 8), 256, 0, st>>>((const bf16*)ws.act[op.in_t], (bf16*)ws.act[op.out_t], (uint8_t*)ws.act[op.mask_t], F, op.C, op.H, op.W);
      }
      else
        pool_fwd_kernel<AT><<<grid_for(total), 256, 0, st>>>((const AT*)ws.act[op.in_t], (AT*)ws.act[op.out_t], F, op.C, op.H, op.W);
      CB_CUDA(cudaGetLastError());
      continue;
    }
    const Layer& L = net->layers[op.layer];
    const Geom& g = L.g;
    int M = F * g.Ho * g.Wo, N = g.Cout, K = g.kh * g.kw * g.Cin;
    const AT* wf = (const AT*)ws.wf + L.wf_off; const float* bias = ws.bias + L.bias_off;
    const AT* skip = L.skip_t >= 0 ? (const AT*)ws.act[L.skip_t] : nullptr;
    if (L.f32_out && L.relu_in && g.kh == 1 && g.kw == 1 && g.H == 1 && g.W == 1 && N <= 32 && !skip) {      // the heads: one warp per frame (its own profile class)
      int rc = launch_heads_sample(std::is_same<AT, bf16>::value ? CB_PREC_BF16_TC : CB_PREC_FP32_REF, ws.act[L.in_t], wf, bias, M, K, N - 1, 0, 0, 0,
                                   (float*)ws.act[L.out_t], nullptr, nullptr, nullptr, st, nullptr, nullptr, taken, n_taken, logp_taken);
      if (rc) return rc;
      continue;
    }
    double in_bytes = (double)F * g.H * g.W * g.Cin * (L.u8_in ? 1 : sizeof(AT));
    ProfScope ps(K_CONV_FWD, st, (std::is_same<AT, bf16>::value && !L.u8_in && !L.f32_out && !L.relu_in && dense_tc_supported(g)) ? 2 : 1, 2.0 * M * N * K, in_bytes + (double)M * N * (L.f32_out ? 4 : sizeof(AT)) * (skip ? 2 : 1) + (double)K * N * sizeof(AT));
    int rc;
    const Op* nxt = oi + 1 < net->fwd.size() ? &net->fwd[oi + 1] : nullptr;
    if (std::is_same<AT, bf16>::value && !L.u8_in && !L.f32_out && !L.relu_in && !L.relu_out && !skip && nxt && nxt->kind == OP_POOL && nxt->in_t == L.out_t &&
        conv_pool_tc_supported(g)) {
      // a stage conv whose only consumer is the max-pool: one kernel, the conv output never reaches HBM (the adjoint needs only the arg-max)
      pool_fused = true;
      rc = launch_conv_pool_tc(g, F, (const bf16*)ws.act[L.in_t], ws.wtc_f + L.wf_off, bias, (bf16*)ws.act[nxt->out_t], (uint8_t*)ws.act[nxt->mask_t], ws.errflag, st);
    } else if (std::is_same<AT, bf16>::value && conv_tc_supported(g) && !L.f32_out && conv_tc_fits(g.H, g.W, g.Cin, g.Cout)) {
      rc = launch_conv_tc(0, F, g.H, g.W, g.Cin, g.Cout, (const bf16*)ws.act[L.in_t], ws.wtc_f + L.wf_off, bias, (const bf16*)skip, nullptr,
                          (bf16*)ws.act[L.out_t], L.relu_in, L.relu_out, ws.errflag, st);
    } else if (std::is_same<AT, bf16>::value && !L.u8_in && !L.f32_out && !L.relu_in && dense_tc_supported(g)) {
      rc = launch_dense_fwd_tc(g, F, (const bf16*)ws.act[L.in_t], ws.wtc_f + L.wf_off, bias, (bf16*)ws.act[L.out_t], ws.partial, ws.errflag, st);
    } else if (std::is_same<AT, bf16>::value && L.u8_in && conv0_tc_supported(g)) {
      const Op* nx = oi + 1 < net->fwd.size() ? &net->fwd[oi + 1] : nullptr;
      pool_fused = nx && nx->kind == OP_POOL && nx->in_t == L.out_t && nx->C % 8 == 0 && g.W % 2 == 0;
      rc = launch_conv0_fwd(g, F, obs, frame_idx, ws.w0img, bias, (bf16*)ws.act[L.out_t], pool_fused ? (bf16*)ws.act[nx->out_t] : nullptr,
                            pool_fused ? (uint8_t*)ws.act[nx->mask_t] : nullptr, ws.errflag, st);
    } else if (L.u8_in) {
      FwdProblem<AT, AT, true> p{M, N, K, K, {g, obs, frame_idx, false}, wf, bias, skip, (AT*)ws.act[L.out_t], 1.0f / 255.0f, L.relu_out};
      rc = launch_gemm(p, 1, st);
    } else if (L.f32_out) {
      FwdProblem<AT, float, false> p{M, N, K, K, {g, ws.act[L.in_t], nullptr, L.relu_in}, wf, bias, skip, (float*)ws.act[L.out_t], 1.0f, L.relu_out};
      rc = launch_gemm(p, 1, st);
    } else {
      FwdProblem<AT, AT, false> p{M, N, K, K, {g, ws.act[L.in_t], nullptr, L.relu_in}, wf, bias, skip, (AT*)ws.act[L.out_t], 1.0f, L.relu_out};
      rc = launch_gemm(p, 1, st);
    }
    if (rc) return rc;
  }
  return CB_OK;
}

int forward(cb_net* net, int prec, const uint8_t* obs, const int32_t* frame_idx, int F, cudaStream_t st, bool skip_heads, const int32_t* taken, int n_taken,
            float* logp_taken) {
  Workspace& ws = net->ws[prec];
  return prec == CB_PREC_FP32_REF ? forward_t<float>(net, ws, obs, frame_idx, F, st, skip_heads, taken, n_taken, logp_taken)
                                  : forward_t<bf16>(net, ws, obs, frame_idx, F, st, skip_heads, taken, n_taken, logp_taken);
}

template <typename AT>
static int backward_t(cb_net* net, Workspace& ws, const uint8_t* obs, const int32_t* frame_idx, int F, float* grad, cudaStream_t st) {
  const Op* fused_pool = nullptr;      // a max-pool adjoint folded into the next (first-layer) weight gradient
  WgradReduceBatch batch;               // tensor-core 3x3 layers: per-layer partial slots, ONE reduction launch after the loop
  size_t tc_off = 0;
  for (size_t oi = 0; oi < net->bwd.size(); ++oi) {
    const Op& op = net->bwd[oi];
    if (op.kind == OP_POOLBWD) {
      if (std::is_same<AT, bf16>::value && op.C % 8 == 0 && oi + 1 < net->bwd.size() && net->bwd[oi + 1].kind == OP_WGRAD) {
        const Layer& NL = net->layers[net->bwd[oi + 1].layer];
        if (NL.u8_in && conv0_tc_supported(NL.g)) { fused_pool = &op; continue; }      // its only consumer gathers through the arg-max itself
      }
      size_t total = (size_t)F * op.H * op.W * op.C;
      ProfScope ps(K_POOL_BWD, st, 1, 0.0, (double)sizeof(AT) * (2.0 * total + (double)F * pool_out(op.H) * pool_out(op.W) * op.C));
      if (std::is_same<AT, bf16>::value && op.C % 8 == 0) {
        const size_t row_bytes = (size_t)op.W * op.C * 2;
        int RB = (int)std::min<size_t>((size_t)op.H, std::max<size_t>(2, (size_t)(40 * 1024) / row_bytes));
        const int nb = (op.H + RB - 1) / RB; RB = (op.H + nb - 1) / nb;
        const size_t smem = (size_t)RB * row_bytes;
        if (smem > 48 * 1024) { int rc = ensure_dyn_smem((const void*)pool_bwd_scatter_kernel, smem); if (rc) return rc; }
        CB_CUDA(launch_pdl(pool_bwd_scatter_kernel, dim3(std::min(F * nb, 148 * 8)), dim3(256), smem, st, (const uint8_t*)ws.act[op.mask_t], (const bf16*)ws.grad[op.dy],
                           (bf16*)ws.grad[op.dx], F, op.C, op.H, op.W, RB, nb));
      } else
        pool_bwd_kernel<AT><<<grid_for(total), 256, 0, st>>>((const AT*)ws.act[op.in_t], (const AT*)ws.grad[op.dy], (AT*)ws.grad[op.dx], F, op.C, op.H, op.W);
      CB_CUDA(cudaGetLastError());
      continue;
    }
    const Layer& L = net->layers[op.layer];
    const Geom& g = L.g;
    if (op.kind == OP_WGRAD) {
      if (std::is_same<AT, bf16>::value && wgrad_tc_supported(g)) {
        const size_t slot = wgrad_tc_partial_elems(g);
        const bool own_slot = tc_off + slot <= ws.partial_tc_elems && batch.n < WGRAD_MAX_JOBS;
        const int jobs_before = batch.n;
        ProfScope ps(K_CONV_WGRAD, st, own_slot ? 1 : 2, 2.0 * 9 * g.Cin * g.Cout * (double)F * g.Ho * g.Wo,
                     2.0 * F * g.H * g.W * (g.Cin + g.Cout) + 4.0 * 9 * (g.Cin + 1) * g.Cout);
        int rc = launch_wgrad_tc(g, L.pm, F, (const bf16*)ws.act[L.in_t], (const bf16*)ws.grad[op.dy], L.relu_in, own_slot ? ws.partial_tc + tc_off : ws.partial, grad,
                                 ws.errflag, st, own_slot ? &batch : nullptr);
        if (rc) return rc;
        if (batch.n > jobs_before) tc_off += slot;      // otherwise the call reduced its partials itself
        continue;
      }
      if (std::is_same<AT, bf16>::value && !L.u8_in && !L.f32_out && !L.relu_in && dense_tc_supported(g)) {
        ProfScope ps(K_CONV_WGRAD, st, 2, 2.0 * g.H * g.W * g.Cin * g.Cout * (double)F, 2.0 * F * (g.H * g.W * g.Cin + g.Cout) + 4.0 * g.H * g.W * g.Cin * g.Cout);
        int rc = launch_dense_wgrad_tc(g, L.pm, F, (const bf16*)ws.act[L.in_t], (const bf16*)ws.grad[op.dy], grad, ws.errflag, st);
        if (rc) return rc;
        continue;
      }
      if (std::is_same<AT, bf16>::value && L.u8_in && conv0_tc_supported(g)) {
        ProfScope ps(K_CONV_WGRAD, st, 2, 2.0 * 9 * g.Cin * g.Cout * (double)F * g.Ho * g.Wo, (double)F * g.H * g.W * (g.Cin + 2.0 * g.Cout));
        int rc = launch_conv0_wgrad(g, L.pm, F, obs, frame_idx, (const bf16*)ws.grad[op.dy],
                                    fused_pool ? (const uint8_t*)ws.act[fused_pool->mask_t] : nullptr, fused_pool ? (const bf16*)ws.grad[fused_pool->dy] : nullptr,
                                    ws.partial, grad, ws.errflag, st);
        fused_pool = nullptr;
        if (rc) return rc;
        continue;
      }
      int Kpix = F * g.Ho * g.Wo, M = g.kh * g.kw * g.Cin + 1, N = g.Cout, splits, kchunk;
      wgrad_split(Kpix, &splits, &kchunk, (long long)((M + 127) / 128) * ((N + 63) / 64));
      double in_bytes = (double)F * g.H * g.W * g.Cin * (L.u8_in ? 1 : sizeof(AT));
      int rc;
      {
      ProfScope ps(K_CONV_WGRAD, st, 1, 2.0 * (M - 1) * N * (double)Kpix, in_bytes + (double)Kpix * N * sizeof(AT) + (double)M * N * 4);
      if (L.u8_in) {
        WgradProblem<AT, AT, true> p{M, N, Kpix, kchunk, {g, obs, frame_idx, false}, (const AT*)ws.grad[op.dy], ws.partial};
        rc = launch_gemm(p, splits, st);
      } else if (L.f32_out && L.relu_in && g.kh == 1 && g.kw == 1 && g.H == 1 && g.W == 1 && N <= 32) {      // the heads
        const int chunk = (F + HEAD_WGRAD_SPLITS - 1) / HEAD_WGRAD_SPLITS;
        splits = (F + chunk - 1) / chunk;
        heads_wgrad_kernel<AT><<<splits, 256, 0, st>>>((const AT*)ws.act[L.in_t], (const AT*)ws.grad[op.dy], ws.partial, F, g.Cin, N, chunk);
        rc = cudaGetLastError() == cudaSuccess ? CB_OK : CB_ECUDA;
      } else {
        WgradProblem<AT, AT, false> p{M, N, Kpix, kchunk, {g, ws.act[L.in_t], nullptr, L.relu_in}, (const AT*)ws.grad[op.dy], ws.partial};
        rc = launch_gemm(p, splits, st);
      }
      }
      if (rc) return rc;
      ProfScope ps2(K_WGRAD_REDUCE, st, 1, 0.0, (double)(splits + 1) * M * N * 4);
      wgrad_reduce_kernel<<<grid_for((size_t)M * N), 256, 0, st>>>(ws.partial, splits, g, L.pm, L.u8_in ? 1.0f / 255.0f : 1.0f, grad);
      CB_CUDA(cudaGetLastError());
    } else {  // OP_DGRAD
      int M = F * g.H * g.W, N = g.Cin, K = g.kh * g.kw * g.Cout;
      // useful MACs of dgrad = those of the forward layer (stride > 1 makes most gathered taps empty)
      ProfScope ps(K_CONV_DGRAD, st, 1, 2.0 * F * g.Ho * g.Wo * (double)g.Cout * g.kh * g.kw * g.Cin,
                   (double)sizeof(AT) * ((double)F * g.Ho * g.Wo * g.Cout + (double)M * N * (1 + (op.mask_t >= 0) + (op.add >= 0)) + (double)K * N));
      if (std::is_same<AT, bf16>::value && conv_tc_supported(g) && conv_tc_fits(g.H, g.W, g.Cout, g.Cin)) {
        int rc = launch_conv_tc(1, F, g.H, g.W, g.Cout, g.Cin, (const bf16*)ws.grad[op.dy], ws.wtc_d + L.wf_off, nullptr,
                                op.mask_t >= 0 ? (const bf16*)ws.act[op.mask_t] : nullptr, op.add >= 0 ? (const bf16*)ws.grad[op.add] : nullptr,
                                (bf16*)ws.grad[op.dx], false, false, ws.errflag, st);
        if (rc) return rc;
        continue;
      }
      if (std::is_same<AT, bf16>::value && !L.f32_out && dense_tc_supported(g) && op.add < 0 && (g.H * g.W * g.Cin) % 16 == 0) {
        int rc = launch_dense_dgrad_tc(g, F, (const bf16*)ws.grad[op.dy], (const bf16*)ws.wf + L.wf_off,
                                       op.mask_t >= 0 ? (const bf16*)ws.act[op.mask_t] : nullptr, (bf16*)ws.grad[op.dx], ws.errflag, st);
        if (rc) return rc;
        continue;
      }
      if (g.Ho == 1 && g.Wo == 1 && g.kh == g.H && g.kw == g.W && g.p == 0) {
        int Nf = g.H * g.W * g.Cin;
        DgradFullProblem<AT> pf{F, Nf, g.Cout, g.Cout, g.Cin, (const AT*)ws.grad[op.dy], (const AT*)ws.wd + L.wd_off,
                                op.mask_t >= 0 ? (const AT*)ws.act[op.mask_t] : nullptr, op.add >= 0 ? (const AT*)ws.grad[op.add] : nullptr, (AT*)ws.grad[op.dx]};
        int rc = launch_gemm(pf, 1, st);
        if (rc) return rc;
        continue;
      }
      DgradProblem<AT> p{M, N, K, K, g, (const AT*)ws.grad[op.dy], (const AT*)ws.wd + L.wd_off,
                         op.mask_t >= 0 ? (const AT*)ws.act[op.mask_t] : nullptr,
                         op.add >= 0 ? (const AT*)ws.grad[op.add] : nullptr, (AT*)ws.grad[op.dx]};
      int rc = launch_gemm(p, 1, st);
      if (rc) return rc;
    }
  }
  if (batch.n > 0) {
    double bytes = 0.0;
    for (int j = 0; j < batch.n; ++j) bytes += 4.0 * (batch.job[j].nctas + 1) * 9 * (batch.job[j].cin_k + 1) * batch.job[j].g.Cout;
    ProfScope ps(K_WGRAD_REDUCE, st, 1, 0.0, bytes);
    int rc = launch_wgrad_reduce_batch(batch, grad, st);
    if (rc) return rc;
  }
  return CB_OK;
}

int backward(cb_net* net, int prec, const uint8_t* obs, const int32_t* frame_idx, int F, float* grad, cudaStream_t st) {
  Workspace& ws = net->ws[prec];
  return prec == CB_PREC_FP32_REF ? backward_t<float>(net, ws, obs, frame_idx, F, grad, st) : backward_t<bf16>(net, ws, obs, frame_idx, F, grad, st);
}

}  // namespace cb
