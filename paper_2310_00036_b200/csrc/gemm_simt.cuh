// Generic SIMT implicit-GEMM (fp32 FFMA, fixed reduction order) used by every linear layer in
// CB_PREC_FP32_REF and as the plain path of CB_PREC_BF16_TC for shapes the tcgen05 kernels do not
// cover.  C[m,n] = sum_k A(m,k) * B(k,n) with A, B fetched through a problem functor:
//   forward : m = (frame, oy, ox)   n = cout   k = (di, dj, cin)
//   dgrad   : m = (frame, y, x)     n = cin    k = (di, dj, cout)
//   wgrad   : m = (di, dj, cin)|bias n = cout  k = (frame, oy, ox), split along k into fixed
//             chunks whose partial sums are added in chunk order by a second kernel
// No atomics anywhere: every output element is written by exactly one thread.
#pragma once
#include "common.cuh"

namespace cb {

__device__ __forceinline__ float ldv(const float* p, size_t i) { return p[i]; }
__device__ __forceinline__ float ldv(const bf16* p, size_t i) { return __bfloat162float(p[i]); }
__device__ __forceinline__ void stv(float* p, size_t i, float v) { p[i] = v; }
__device__ __forceinline__ void stv(bf16* p, size_t i, float v) { p[i] = __float2bfloat16_rn(v); }

// input element of a conv layer at (frame f, output pixel (oy,ox), tap (di,dj), channel c)
template <typename AT, bool U8>
struct ConvInput {
  Geom g; const void* x; const int32_t* frame_idx; bool relu;
  __device__ __forceinline__ float at(int f, int oy, int ox, int di, int dj, int c) const {
    int iy = oy * g.s + di - g.p, ix = ox * g.s + dj - g.p;
    if ((unsigned)iy >= (unsigned)g.H || (unsigned)ix >= (unsigned)g.W) return 0.f;
    if (U8) {
      size_t fr = frame_idx ? (size_t)frame_idx[f] : (size_t)f;
      return (float)((const uint8_t*)x)[((fr * g.Cin + c) * g.H + iy) * g.W + ix];   // NCHW uint8, raw integer
    } else {
      float v = ldv((const AT*)x, (((size_t)f * g.H + iy) * g.W + ix) * g.Cin + c);
      return relu ? fmaxf(v, 0.f) : v;
    }
  }
};

struct Pix { int f, oy, ox; bool ok; };
struct Tap { int di, dj, c; bool ok; };

template <typename AT, typename OT, bool U8>
struct FwdProblem {
  static constexpr bool A_K_FAST = true;
  int M, N, K, kchunk;
  ConvInput<AT, U8> in; const AT* w; const float* bias; const AT* skip; OT* y; float in_scale; bool relu_out;
  typedef Pix RowA; typedef Tap ColA;
  __device__ RowA rowA(int m) const { Pix r; r.ok = m < M; int q = in.g.Ho * in.g.Wo; r.f = m / q; int rem = m - r.f * q; r.oy = rem / in.g.Wo; r.ox = rem - r.oy * in.g.Wo; return r; }
  __device__ ColA colA(int k) const { Tap t; t.ok = k < K; t.c = k % in.g.Cin; int q = k / in.g.Cin; t.dj = q % in.g.kw; t.di = q / in.g.kw; return t; }
  __device__ float loadA(const RowA& r, const ColA& t) const { return (r.ok && t.ok) ? in.at(r.f, r.oy, r.ox, t.di, t.dj, t.c) : 0.f; }
  __device__ float loadB(int k, int n) const { return (k < K && n < N) ? ldv(w, (size_t)k * N + n) : 0.f; }
  __device__ void store(int m, int n, float acc, int) const {
    float v = acc * in_scale + bias[n];
    size_t i = (size_t)m * N + n;
    if (skip) v += ldv(skip, i);
    if (relu_out) v = fmaxf(v, 0.f);
    stv(y, i, v);
  }
};

template <typename AT>
struct DgradProblem {
  static constexpr bool A_K_FAST = true;
  int M, N, K, kchunk;   // M = F*H*W, N = Cin, K = kh*kw*Cout
  Geom g; const AT* dy; const AT* w;   // w packed [(di,dj,o)][c]
  const AT* mask; const AT* add; AT* dx;
  struct RowA { int f, y, x; bool ok; };
  typedef Tap ColA;   // c field holds the output channel o
  __device__ RowA rowA(int m) const { RowA r; r.ok = m < M; int q = g.H * g.W; r.f = m / q; int rem = m - r.f * q; r.y = rem / g.W; r.x = rem - r.y * g.W; return r; }
  __device__ ColA colA(int k) const { Tap t; t.ok = k < K; t.c = k % g.Cout; int q = k / g.Cout; t.dj = q % g.kw; t.di = q / g.kw; return t; }
  __device__ float loadA(const RowA& r, const ColA& t) const {
    if (!(r.ok && t.ok)) return 0.f;
    int ty = r.y + g.p - t.di, tx = r.x + g.p - t.dj;
    if (ty < 0 || tx < 0) return 0.f;
    int oy = ty / g.s, ox = tx / g.s;
    if (oy * g.s != ty || ox * g.s != tx || oy >= g.Ho || ox >= g.Wo) return 0.f;
    return ldv(dy, (((size_t)r.f * g.Ho + oy) * g.Wo + ox) * g.Cout + t.c);
  }
  __device__ float loadB(int k, int n) const { return (k < K && n < N) ? ldv(w, (size_t)k * N + n) : 0.f; }
  __device__ void store(int m, int n, float acc, int) const {
    size_t i = (size_t)m * N + n; float v = acc;
    if (mask && !(ldv(mask, i) > 0.f)) v = 0.f;     // ReLU'(x <= 0) = 0 (A11)
    if (add) v += ldv(add, i);
    stv(dx, i, v);
  }
};

// dgrad of a layer whose kernel covers its whole input (fc, heads): a plain GEMM
//   dx[f, (y,x,c)] = sum_o dy[f,o] * w[o,c,y,x],   B read from the dgrad pack Wd[(y,x,o)][c]
template <typename AT>
struct DgradFullProblem {
  static constexpr bool A_K_FAST = true;
  int M, N, K, kchunk;   // M = F, N = H*W*Cin, K = Cout
  int Cin; const AT* dy; const AT* wd; const AT* mask; const AT* add; AT* dx;
  struct RowA { int m; bool ok; };
  struct ColA { int k; bool ok; };
  __device__ RowA rowA(int m) const { return {m, m < M}; }
  __device__ ColA colA(int k) const { return {k, k < K}; }
  __device__ float loadA(const RowA& r, const ColA& c) const { return (r.ok && c.ok) ? ldv(dy, (size_t)r.m * K + c.k) : 0.f; }
  __device__ float loadB(int k, int n) const {
    if (k >= K || n >= N) return 0.f;
    int t = n / Cin, c = n - t * Cin;
    return ldv(wd, ((size_t)t * K + k) * Cin + c);
  }
  __device__ void store(int m, int n, float acc, int) const {
    size_t i = (size_t)m * N + n; float v = acc;
    if (mask && !(ldv(mask, i) > 0.f)) v = 0.f;
    if (add) v += ldv(add, i);
    stv(dx, i, v);
  }
};

template <typename AT, typename GT, bool U8>
struct WgradProblem {
  static constexpr bool A_K_FAST = false;
  int M, N, K, kchunk;   // M = kh*kw*Cin + 1 (last row = bias), N = Cout, K = F*Ho*Wo
  ConvInput<AT, U8> in; const GT* dy; float* partial;
  typedef Tap RowA; typedef Pix ColA;
  __device__ RowA rowA(int m) const { Tap t; t.ok = m < M; t.c = m % in.g.Cin; int q = m / in.g.Cin; t.dj = q % in.g.kw; t.di = q / in.g.kw; return t; }   // bias row: di == kh
  __device__ ColA colA(int k) const { Pix r; r.ok = k < K; int q = in.g.Ho * in.g.Wo; r.f = k / q; int rem = k - r.f * q; r.oy = rem / in.g.Wo; r.ox = rem - r.oy * in.g.Wo; return r; }
  __device__ float loadA(const RowA& t, const ColA& r) const {
    if (!(r.ok && t.ok)) return 0.f;
    if (t.di >= in.g.kh) return 1.f;                 // bias row: db[o] = sum_pixels dy
    return in.at(r.f, r.oy, r.ox, t.di, t.dj, t.c);
  }
  __device__ float loadB(int k, int n) const { return (k < K && n < N) ? ldv(dy, (size_t)k * N + n) : 0.f; }
  __device__ void store(int m, int n, float acc, int split) const { partial[((size_t)split * M + m) * N + n] = acc; }
};

// BM = 128 rows, BN in {16,32,64} columns, BK = 16; 256 threads as 16 (n) x 16 (m), each 8 x BN/16.
template <int BN, class P>
__global__ void __launch_bounds__(256) gemm_simt_kernel(const P p) {
  constexpr int BM = 128, BK = 16, TM = 8, TN = BN / 16;
  __shared__ float As[BK][BM + 4];
  __shared__ float Bs[BK][BN + 4];
  const int t = threadIdx.x, tx = t & 15, ty = t >> 4;
  const int m0 = blockIdx.x * BM, n0 = blockIdx.y * BN, split = blockIdx.z;
  const int kbeg = split * p.kchunk, kend = min(p.K, kbeg + p.kchunk);
  float acc[TM][TN];
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int j = 0; j < TN; ++j) acc[i][j] = 0.f;

  typename P::RowA rows[P::A_K_FAST ? 8 : 1];
  if (P::A_K_FAST) {
#pragma unroll
    for (int i = 0; i < 8; ++i) rows[i] = p.rowA(m0 + (t >> 4) + 16 * i);
  } else {
    rows[0] = p.rowA(m0 + (t & 127));
  }

  for (int k0 = kbeg; k0 < kend; k0 += BK) {
    if (P::A_K_FAST) {
      int kk = t & 15; int k = k0 + kk;
      typename P::ColA col = p.colA(k < kend ? k : p.K);
#pragma unroll
      for (int i = 0; i < 8; ++i) As[kk][(t >> 4) + 16 * i] = p.loadA(rows[i], col);
    } else {
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        int kk = (t >> 7) + 2 * i; int k = k0 + kk;
        typename P::ColA col = p.colA(k < kend ? k : p.K);
        As[kk][t & 127] = p.loadA(rows[0], col);
      }
    }
#pragma unroll
    for (int i = 0; i < BN / 16; ++i) {
      int e = t + 256 * i; int kk = e / BN, nn = e % BN; int k = k0 + kk;
      Bs[kk][nn] = (k < kend) ? p.loadB(k, n0 + nn) : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < BK; ++kk) {
      float a[TM], b[TN];
#pragma unroll
      for (int i = 0; i < TM; ++i) a[i] = As[kk][ty * TM + i];
#pragma unroll
      for (int j = 0; j < TN; ++j) b[j] = Bs[kk][tx + 16 * j];
#pragma unroll
      for (int i = 0; i < TM; ++i)
#pragma unroll
        for (int j = 0; j < TN; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < TM; ++i) {
    int m = m0 + ty * TM + i;
    if (m >= p.M) continue;
#pragma unroll
    for (int j = 0; j < TN; ++j) {
      int n = n0 + tx + 16 * j;
      if (n < p.N) p.store(m, n, acc[i][j], split);
    }
  }
}

template <class P>
int launch_gemm(const P& p, int splits, cudaStream_t st) {
  if (p.M <= 0 || p.N <= 0) return CB_OK;
  dim3 block(256);
  unsigned gm = (unsigned)((p.M + 127) / 128);
  if (p.N <= 16) { dim3 grid(gm, 1, splits); gemm_simt_kernel<16, P><<<grid, block, 0, st>>>(p); }
  else if (p.N <= 32) { dim3 grid(gm, 1, splits); gemm_simt_kernel<32, P><<<grid, block, 0, st>>>(p); }
  else { dim3 grid(gm, (unsigned)((p.N + 63) / 64), splits); gemm_simt_kernel<64, P><<<grid, block, 0, st>>>(p); }
  CB_CUDA(cudaGetLastError());
  return CB_OK;
}

}  // namespace cb
