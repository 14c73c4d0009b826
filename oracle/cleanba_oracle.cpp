// =============================================================================================
// cleanba_oracle.cpp -- CPU ORACLE for the Cleanba agent hot path.  TEST INFRASTRUCTURE ONLY.
//
// This file is the plain, slow, single-threaded definition of what the CUDA library under
// paper_2310_00036_b200/csrc must compute.  It shares no code, header, table or constant
// generator with that library and neither includes the other.  Only tests/, bench.py's
// cpu_baseline / --impl reference leg and __graft_entry__.smoke() may load it.
//
// Arithmetic: fp32 inputs and parameters, every sum and every transcendental in fp64, results
// rounded to fp32 only where the C ABI exposes fp32 (logits, values, params, Adam state, stats).
//
// Citations are PAPER.md:<line> (/root/reference/PAPER.md, arXiv 2310.00036) or a reading
// "A<n>" listed in DESIGN.md section 3 where the paper is silent.
//
// Pin status (tests/test_oracle_*.py, all `-m "not gpu"`):
//   network forward/backward ... pinned: torch-CPU fp64 conv2d/max_pool2d/linear + autograd,
//                                 brute-force finite differences, hand-built pool tie case
//   softmax / entropy ........... pinned: identities (sum p = 1, H(uniform)=log A, shift invariance)
//   Philox4x32-10 ............... pinned: cuRAND host generator (library) on 1e6 counters
//   fixed-op log / Gumbel ....... pinned: libm log over all 2^24 uniforms, chi^2 vs softmax
//   V-trace ..................... pinned: n-step-return closed form, c_bar=0, GAE cross-pin, T=1, the lambda mix of q_t
//                                 (on-policy pgadv = GAE(lambda) by double sum), the off-policy definition as an
//                                 explicit double sum with three different thresholds (rho_bar, c_bar, rho_pg_bar)
//   GAE ......................... pinned: lambda=1 brute-force discounted return, lambda=0
//   IMPALA / PPO losses ......... pinned: finite differences, ratio-1 invariants, sign tests
//   clip + Adam ................. pinned: first-step closed form, constant-gradient closed form
//   clip + RMSprop (A22) ........ pinned: first-step and constant-gradient closed forms, lr = 0
//   env-split minibatches (A21) . pinned: mb = 1 identity, equality with per-group single steps run by hand
//   permutation ................. pinned: bijection + brute-force reference of the index rule
//   behaviour values (A3b) ...... pinned: step with the oracle's own recomputed (fp32-rounded) values == hand-composed
//                                 GAE + minibatch updates; values of a different policy change the targets only
//   PPO epoch counter (A23) ..... pinned: a second call continues the permutation epochs where the first stopped
// =============================================================================================
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include <algorithm>
#include <limits>

extern "C" {

typedef struct {
  int kind;          // 0 = Nature-CNN (BASELINE.json configs[0]), 1 = IMPALA-ResNet
  int in_c, in_h, in_w;   // 4, 84, 84 for Atari; smaller for tiny test nets
  int channels[3];
  int fc;
  int n_actions;     // 18, "full action space"
} orc_arch;

typedef struct {
  int algo;          // 0 IMPALA, 1 PPO
  int T, B;
  double gamma, lambda_;
  double rho_bar, c_bar, rho_pg_bar;              // Table 3
  double clip_eps; int epochs, minibatches, norm_adv; uint64_t perm_seed;   // Table 2
  double vf_coef, ent_coef;                       // c1, c2
  double lr, beta1, beta2, adam_eps, max_grad_norm;
  int loss_reduction;                             // 0 mean, 1 sum (reading A4)
  int optimizer;                                  // 0 Adam (A12), 1 RMSprop (Table 3; reading A22)
  double rms_decay, rms_eps;                      // 0.99, 0.01
} orc_hparams;

enum { ORC_N_STATS = 8 };  // loss, pg_loss, v_loss, entropy, grad_norm, approx_kl, clip_frac, mean_rho

}  // extern "C"

namespace {

typedef std::vector<double> vec;

// ---------------------------------------------------------------------------------------------
// Shapes.  Reading A10: conv3x3 stride 1 zero pad 1; max-pool 3x3 stride 2 "SAME" in the XLA
// sense (the paper's stack is JAX): out = ceil(H/2), total pad =
// max((out-1)*2+3-H, 0), pad_lo = floor(total/2); padded cells never win.
// ---------------------------------------------------------------------------------------------
int pool_out(int h) { return (h + 1) / 2; }
int pool_pad_lo(int h) { int o = pool_out(h); int tot = std::max((o - 1) * 2 + 3 - h, 0); return tot / 2; }
int conv_out(int h, int k, int s, int pad) { return (h + 2 * pad - k) / s + 1; }

struct LayerSpec { int cin, cout, k, stride, pad; };

// Parameter layout (reading §8(b) "Layouts"): stage/layer order, weight then bias; conv weights
// [Cout,Cin,kh,kw]; FC weights [out,in] with `in` flattened in (C,H,W) order.
struct Layout {
  std::vector<LayerSpec> convs;   // in forward order
  std::vector<size_t> conv_w, conv_b;
  size_t fc_w, fc_b, pi_w, pi_b, v_w, v_b, total;
  int fc_in, feat_c, feat_h, feat_w;
};

Layout make_layout(const orc_arch& a) {
  Layout L; size_t off = 0; int h = a.in_h, w = a.in_w, c = a.in_c;
  auto add_conv = [&](int cout, int k, int s, int pad) {
    L.convs.push_back({c, cout, k, s, pad});
    L.conv_w.push_back(off); off += (size_t)cout * c * k * k;
    L.conv_b.push_back(off); off += cout;
    h = conv_out(h, k, s, pad); w = conv_out(w, k, s, pad); c = cout;
  };
  if (a.kind == 0) {            // conv 8x8s4, 4x4s2, 3x3s1, all VALID (BASELINE.json configs[0])
    add_conv(a.channels[0], 8, 4, 0);
    add_conv(a.channels[1], 4, 2, 0);
    add_conv(a.channels[2], 3, 1, 0);
  } else {                      // 3 x [conv3x3, maxpool3x3s2, 2 residual blocks] (configs[1])
    for (int s = 0; s < 3; ++s) {
      add_conv(a.channels[s], 3, 1, 1);
      h = pool_out(h); w = pool_out(w);
      for (int i = 0; i < 4; ++i) add_conv(a.channels[s], 3, 1, 1);
    }
  }
  L.feat_c = c; L.feat_h = h; L.feat_w = w; L.fc_in = c * h * w;
  L.fc_w = off; off += (size_t)a.fc * L.fc_in;
  L.fc_b = off; off += a.fc;
  L.pi_w = off; off += (size_t)a.n_actions * a.fc;
  L.pi_b = off; off += a.n_actions;
  L.v_w = off; off += a.fc;
  L.v_b = off; off += 1;
  L.total = off;
  return L;
}

// ---------------------------------------------------------------------------------------------
// O1 primitives.  Convolution is cross-correlation with zero padding:
//   y[o,i,j] = b[o] + sum_{c,di,dj} w[o,c,di,dj] * x[c, i*s+di-p, j*s+dj-p]
// ---------------------------------------------------------------------------------------------
void conv_fwd(const vec& x, int cin, int H, int W, const double* w, const double* b,
              int cout, int k, int s, int p, vec& y) {
  int Ho = conv_out(H, k, s, p), Wo = conv_out(W, k, s, p);
  y.assign((size_t)cout * Ho * Wo, 0.0);
  for (int o = 0; o < cout; ++o) {
    double* yo = &y[(size_t)o * Ho * Wo];
    for (int q = 0; q < Ho * Wo; ++q) yo[q] = b[o];
    for (int c = 0; c < cin; ++c)
      for (int di = 0; di < k; ++di)
        for (int dj = 0; dj < k; ++dj) {
          double wv = w[(((size_t)o * cin + c) * k + di) * k + dj];
          for (int i = 0; i < Ho; ++i) {
            int yi = i * s + di - p; if (yi < 0 || yi >= H) continue;
            const double* xr = &x[((size_t)c * H + yi) * W];
            for (int j = 0; j < Wo; ++j) {
              int xj = j * s + dj - p; if (xj < 0 || xj >= W) continue;
              yo[(size_t)i * Wo + j] += wv * xr[xj];
            }
          }
        }
  }
}

// Adjoint of conv_fwd (O8): dx (optional), dw += , db += .
void conv_bwd(const vec& x, int cin, int H, int W, const double* w, int cout, int k, int s, int p,
              const vec& dy, vec* dx, double* dw, double* db) {
  int Ho = conv_out(H, k, s, p), Wo = conv_out(W, k, s, p);
  if (dx) dx->assign((size_t)cin * H * W, 0.0);
  for (int o = 0; o < cout; ++o) {
    const double* dyo = &dy[(size_t)o * Ho * Wo];
    double sb = 0.0; for (int q = 0; q < Ho * Wo; ++q) sb += dyo[q];
    db[o] += sb;
    for (int c = 0; c < cin; ++c)
      for (int di = 0; di < k; ++di)
        for (int dj = 0; dj < k; ++dj) {
          size_t wi = (((size_t)o * cin + c) * k + di) * k + dj;
          double wv = w[wi], acc = 0.0;
          for (int i = 0; i < Ho; ++i) {
            int yi = i * s + di - p; if (yi < 0 || yi >= H) continue;
            const double* xr = &x[((size_t)c * H + yi) * W];
            double* dxr = dx ? &(*dx)[((size_t)c * H + yi) * W] : nullptr;
            for (int j = 0; j < Wo; ++j) {
              int xj = j * s + dj - p; if (xj < 0 || xj >= W) continue;
              double g = dyo[(size_t)i * Wo + j];
              acc += g * xr[xj];
              if (dxr) dxr[xj] += g * wv;
            }
          }
          dw[wi] += acc;
        }
  }
}

// Max-pool 3x3 stride 2, XLA-SAME padding (A10); argmax = FIRST maximum in row-major window
// order (A11), stored as flat input index for the adjoint.
void pool_fwd(const vec& x, int C, int H, int W, vec& y, std::vector<int>& arg) {
  int Ho = pool_out(H), Wo = pool_out(W), pl_h = pool_pad_lo(H), pl_w = pool_pad_lo(W);
  y.assign((size_t)C * Ho * Wo, 0.0); arg.assign((size_t)C * Ho * Wo, -1);
  for (int c = 0; c < C; ++c)
    for (int i = 0; i < Ho; ++i)
      for (int j = 0; j < Wo; ++j) {
        double best = -std::numeric_limits<double>::infinity(); int bi = -1;
        for (int di = 0; di < 3; ++di)
          for (int dj = 0; dj < 3; ++dj) {
            int yi = i * 2 + di - pl_h, xj = j * 2 + dj - pl_w;
            if (yi < 0 || yi >= H || xj < 0 || xj >= W) continue;
            int idx = (c * H + yi) * W + xj;
            if (x[idx] > best) { best = x[idx]; bi = idx; }   // strict > keeps the first maximum
          }
        y[((size_t)c * Ho + i) * Wo + j] = best; arg[((size_t)c * Ho + i) * Wo + j] = bi;
      }
}

void relu(const vec& x, vec& y) { y.resize(x.size()); for (size_t i = 0; i < x.size(); ++i) y[i] = x[i] > 0.0 ? x[i] : 0.0; }
// ReLU'(x <= 0) = 0 (A11)
void relu_bwd(const vec& x, vec& g) { for (size_t i = 0; i < x.size(); ++i) if (!(x[i] > 0.0)) g[i] = 0.0; }

// ---------------------------------------------------------------------------------------------
// Network forward with a tape (one frame).  PAPER.md:181 (IMPALA ResNet by citation),
// BASELINE.json configs[0] (Nature-CNN), reading O1.
// ---------------------------------------------------------------------------------------------
struct Tape {
  std::vector<vec> conv_in;      // input of each conv (post-ReLU where a ReLU precedes it)
  std::vector<vec> pre;          // pre-activation tensors whose sign gates a ReLU
  std::vector<std::vector<int>> pool_arg;
  std::vector<int> pool_in_size;
  vec feat_pre, feat, hid_pre, hid;
};

void net_forward(const orc_arch& a, const Layout& L, const double* P, const uint8_t* obs,
                 double* logits, double* value, Tape* tp) {
  int H = a.in_h, W = a.in_w, C = a.in_c;
  vec x((size_t)C * H * W);
  for (size_t i = 0; i < x.size(); ++i) x[i] = (double)obs[i] / 255.0;        // O1: x = u8/255
  Tape local; Tape& t = tp ? *tp : local;
  t.conv_in.clear(); t.pre.clear(); t.pool_arg.clear(); t.pool_in_size.clear();
  int li = 0; vec y, r;
  auto conv = [&](const vec& in, vec& out) {
    const LayerSpec& s = L.convs[li];
    conv_fwd(in, s.cin, H, W, P + L.conv_w[li], P + L.conv_b[li], s.cout, s.k, s.stride, s.pad, out);
    t.conv_in.push_back(in);
    H = conv_out(H, s.k, s.stride, s.pad); W = conv_out(W, s.k, s.stride, s.pad); C = s.cout; ++li;
  };
  if (a.kind == 0) {
    for (int i = 0; i < 3; ++i) { conv(x, y); t.pre.push_back(y); relu(y, x); }
    t.feat_pre = t.pre.back(); t.feat = x;            // already ReLU'd
  } else {
    for (int s = 0; s < 3; ++s) {
      conv(x, y);
      std::vector<int> arg; vec p;
      t.pool_in_size.push_back((int)y.size());
      pool_fwd(y, C, H, W, p, arg); t.pool_arg.push_back(arg);
      H = pool_out(H); W = pool_out(W);
      for (int b = 0; b < 2; ++b) {       // x <- x + conv(relu(conv(relu(x))))
        vec h1, h2;
        t.pre.push_back(p); relu(p, r); conv(r, h1);
        t.pre.push_back(h1); relu(h1, r); conv(r, h2);
        for (size_t i = 0; i < p.size(); ++i) p[i] += h2[i];
      }
      x = p;
    }
    t.feat_pre = x; relu(x, t.feat);
  }
  // trunk: flatten (C,H,W) -> FC -> ReLU; heads linear from the same hidden vector (O1)
  int K = L.fc_in;
  t.hid_pre.assign(a.fc, 0.0);
  for (int o = 0; o < a.fc; ++o) {
    double s = P[L.fc_b + o]; const double* wr = P + L.fc_w + (size_t)o * K;
    for (int k = 0; k < K; ++k) s += wr[k] * t.feat[k];
    t.hid_pre[o] = s;
  }
  relu(t.hid_pre, t.hid);
  for (int i = 0; i < a.n_actions; ++i) {
    double s = P[L.pi_b + i]; const double* wr = P + L.pi_w + (size_t)i * a.fc;
    for (int k = 0; k < a.fc; ++k) s += wr[k] * t.hid[k];
    logits[i] = s;
  }
  double s = P[L.v_b];
  for (int k = 0; k < a.fc; ++k) s += P[L.v_w + k] * t.hid[k];
  *value = s;
}

// Adjoint of net_forward for one frame; accumulates into G[L.total] (O8).
void net_backward(const orc_arch& a, const Layout& L, const double* P, const Tape& t,
                  const double* dlogits, double dvalue, double* G) {
  int A = a.n_actions, F = a.fc, K = L.fc_in;
  vec dhid(F, 0.0);
  for (int i = 0; i < A; ++i) {
    G[L.pi_b + i] += dlogits[i];
    for (int k = 0; k < F; ++k) { G[L.pi_w + (size_t)i * F + k] += dlogits[i] * t.hid[k]; dhid[k] += dlogits[i] * P[L.pi_w + (size_t)i * F + k]; }
  }
  G[L.v_b] += dvalue;
  for (int k = 0; k < F; ++k) { G[L.v_w + k] += dvalue * t.hid[k]; dhid[k] += dvalue * P[L.v_w + k]; }
  relu_bwd(t.hid_pre, dhid);
  vec dfeat(K, 0.0);
  for (int o = 0; o < F; ++o) {
    G[L.fc_b + o] += dhid[o];
    double* gw = G + L.fc_w + (size_t)o * K; const double* wr = P + L.fc_w + (size_t)o * K;
    for (int k = 0; k < K; ++k) { gw[k] += dhid[o] * t.feat[k]; dfeat[k] += dhid[o] * wr[k]; }
  }
  relu_bwd(t.feat_pre, dfeat);
  // spatial sizes of every conv input, replayed forward
  std::vector<int> Hs, Ws; { int h = a.in_h, w = a.in_w;
    if (a.kind == 0) { for (int i = 0; i < 3; ++i) { Hs.push_back(h); Ws.push_back(w); const LayerSpec& s = L.convs[i]; h = conv_out(h, s.k, s.stride, s.pad); w = conv_out(w, s.k, s.stride, s.pad); } }
    else { for (int s = 0; s < 3; ++s) { Hs.push_back(h); Ws.push_back(w); h = pool_out(h); w = pool_out(w); for (int i = 0; i < 4; ++i) { Hs.push_back(h); Ws.push_back(w); } } } }
  auto conv_b = [&](int li, const vec& dy, vec* dx) {
    const LayerSpec& s = L.convs[li];
    conv_bwd(t.conv_in[li], s.cin, Hs[li], Ws[li], P + L.conv_w[li], s.cout, s.k, s.stride, s.pad, dy, dx,
             G + L.conv_w[li], G + L.conv_b[li]);
  };
  if (a.kind == 0) {
    vec d = dfeat;                         // gradient w.r.t. relu(conv3) output, already gated above
    for (int li = 2; li >= 0; --li) {
      if (li < 2) relu_bwd(t.pre[li], d);
      vec dx; conv_b(li, d, li > 0 ? &dx : nullptr); d.swap(dx);
    }
  } else {
    vec d = dfeat;                         // gradient w.r.t. stage-3 output (pre final ReLU, gated above)
    for (int s = 2; s >= 0; --s) {
      for (int b = 1; b >= 0; --b) {
        int li2 = s * 5 + 1 + b * 2 + 1, li1 = li2 - 1, pi = (s * 2 + b) * 2;
        vec dr2, dr1;
        conv_b(li2, d, &dr2); relu_bwd(t.pre[pi + 1], dr2);
        conv_b(li1, dr2, &dr1); relu_bwd(t.pre[pi], dr1);
        for (size_t i = 0; i < d.size(); ++i) d[i] += dr1[i];   // residual: identity path + block path
      }
      vec dc(t.pool_in_size[s], 0.0);
      const std::vector<int>& arg = t.pool_arg[s];
      for (size_t i = 0; i < arg.size(); ++i) dc[arg[i]] += d[i];  // whole gradient to the arg-max (A11)
      vec dx; conv_b(s * 5, dc, s > 0 ? &dx : nullptr); d.swap(dx);
    }
  }
}

// ---------------------------------------------------------------------------------------------
// O2 distribution math: lse = max + log sum exp(l - max); log p = l - lse; H = -sum p log p.
// ---------------------------------------------------------------------------------------------
void log_softmax(const double* l, int A, double* logp) {
  double m = l[0]; for (int i = 1; i < A; ++i) m = std::max(m, l[i]);
  double s = 0.0; for (int i = 0; i < A; ++i) s += std::exp(l[i] - m);
  double lse = m + std::log(s);
  for (int i = 0; i < A; ++i) logp[i] = l[i] - lse;
}
double entropy_of(const double* logp, int A) { double h = 0.0; for (int i = 0; i < A; ++i) h -= std::exp(logp[i]) * logp[i]; return h; }

// ---------------------------------------------------------------------------------------------
// A9: Philox4x32-10 (Salmon et al. 2011, the counter-based generator BASELINE.json names).
// ---------------------------------------------------------------------------------------------
void philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
  uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3], k0 = key_in[0], k1 = key_in[1];
  for (int r = 0; r < 10; ++r) {
    uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1, n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// A9: natural log by a FIXED sequence of IEEE-754 binary64 operations (integer exponent split,
// one division, Horner with fma), so an independent implementation rounds identically.
//   x = m * 2^e, m in (sqrt(1/2), sqrt(2)];  s = (m-1)/(m+1);  log m = 2 atanh(s) = s * sum_k c_k s^(2k),
//   c_k = 2/(2k+1) rounded to binary64, k = 0..12;  log x = e*LN2_HI + (e*LN2_LO + log m).
// Valid for positive normal x (all this path ever sees).
double fixed_log(double x) {
  static const double C[13] = {
      2.0, 0x1.5555555555555p-1, 0x1.999999999999ap-2, 0x1.2492492492492p-2, 0x1.c71c71c71c71cp-3,
      0x1.745d1745d1746p-3, 0x1.3b13b13b13b14p-3, 0x1.1111111111111p-3, 0x1.e1e1e1e1e1e1ep-4,
      0x1.af286bca1af28p-4, 0x1.8618618618618p-4, 0x1.642c8590b2164p-4, 0x1.47ae147ae147bp-4};
  const double LN2_HI = 0x1.62e42fee00000p-1, LN2_LO = 0x1.a39ef35793c76p-33;
  uint64_t bits; std::memcpy(&bits, &x, 8);
  int e = (int)((bits >> 52) & 0x7ff) - 1023;
  bits = (bits & 0x000fffffffffffffULL) | 0x3ff0000000000000ULL;
  double m; std::memcpy(&m, &bits, 8);
  if (m > 0x1.6a09e667f3bcdp+0) { m = m * 0.5; e += 1; }
  double s = (m - 1.0) / (m + 1.0);
  double z = s * s;
  double p = C[12];
  for (int k = 11; k >= 0; --k) p = std::fma(p, z, C[k]);
  double lm = s * p;
  double ed = (double)e;
  return std::fma(ed, LN2_HI, std::fma(ed, LN2_LO, lm));
}

// u = ((x >> 8) + 0.5) * 2^-24 in (0,1), exact in binary64;  g = -log(-log u), rounded once to fp32.
float gumbel_from_u32(uint32_t x) {
  double u = ((double)(x >> 8) + 0.5) * 0x1p-24;
  double g = -fixed_log(-fixed_log(u));
  return (float)g;
}

// O3 / A9: a = argmax_i (fp32 logit_i + fp32 gumbel_i) in fp32, lowest index on ties.
// counter = (env, step_lo, step_hi, j), key = (seed_lo, seed_hi); word w of block j -> action 4j+w.
int sample_action(const float* logits, int A, uint64_t seed, uint64_t step, uint32_t env) {
  uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  int best = 0; float bs = 0.f;
  for (int j = 0; j * 4 < A; ++j) {
    uint32_t ctr[4] = {env, (uint32_t)step, (uint32_t)(step >> 32), (uint32_t)j}, r[4];
    philox4x32_10(ctr, key, r);
    for (int w = 0; w < 4 && 4 * j + w < A; ++w) {
      int i = 4 * j + w;
      float sc = logits[i] + gumbel_from_u32(r[w]);
      if (i == 0 || sc > bs) { bs = sc; best = i; }
    }
  }
  return best;
}

// A17: per-epoch Fisher-Yates permutation of N flat indices (flat index = t*B + b).
// Draw q = 0,1,... is word q%4 of Philox block counter (q/4, epoch, 0, 0x5045524D), key = perm_seed;
// for i = N-1 down to 1: j = (x * (i+1)) >> 32 with x the next draw; swap(perm[i], perm[j]).
void permutation(uint64_t seed, uint32_t epoch, int N, int32_t* perm) {
  uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  for (int i = 0; i < N; ++i) perm[i] = i;
  uint32_t r[4]; int q = 0;
  for (int i = N - 1; i >= 1; --i, ++q) {
    if (q % 4 == 0) { uint32_t ctr[4] = {(uint32_t)(q / 4), epoch, 0u, 0x5045524Du}; philox4x32_10(ctr, key, r); }
    uint32_t j = (uint32_t)(((uint64_t)r[q % 4] * (uint64_t)(i + 1)) >> 32);
    std::swap(perm[i], perm[j]);
  }
}

// ---------------------------------------------------------------------------------------------
// O4 V-trace (PAPER.md:370, 414 point at rlax; equations are Espeholt et al. 2018 with lambda
// mixing, reading A2).  dones[t] = 1 <=> the step taken at t ended the episode (A1).
//   disc_t = gamma (1 - d_t);  w_t = exp(log pi(a_t) - log mu(a_t));  rho_t = min(rho_bar, w_t)
//   c_t = lambda min(c_bar, w_t);  delta_t = rho_t (r_t + disc_t V_{t+1} - V_t)
//   acc_T = 0;  acc_t = delta_t + disc_t c_t acc_{t+1};  vs_t = V_t + acc_t;  vs_T = V_T
//   q_t = r_t + disc_t (lambda vs_{t+1} + (1-lambda) V_{t+1});  pgadv_t = min(rho_pg_bar, w_t)(q_t - V_t)
// ---------------------------------------------------------------------------------------------
void vtrace(int T, int B, const double* V, const double* r, const uint8_t* d, const double* logpi,
            const double* logmu, double gamma, double lam, double rho_bar, double c_bar, double rho_pg_bar,
            double* vs, double* pgadv, double* rho_out) {
  for (int b = 0; b < B; ++b) {
    double acc = 0.0, vs_next = V[(size_t)T * B + b];
    for (int t = T - 1; t >= 0; --t) {
      size_t i = (size_t)t * B + b;
      double disc = gamma * (1.0 - (double)d[i]);
      double w = std::exp(logpi[i] - logmu[i]);
      double rho = std::min(rho_bar, w), c = lam * std::min(c_bar, w);
      double Vn = V[i + B];
      double delta = rho * (r[i] + disc * Vn - V[i]);
      acc = delta + disc * c * acc;
      double q = r[i] + disc * (lam * vs_next + (1.0 - lam) * Vn);
      pgadv[i] = std::min(rho_pg_bar, w) * (q - V[i]);
      vs[i] = V[i] + acc; vs_next = vs[i];
      if (rho_out) rho_out[i] = rho;
    }
  }
}

// O6 GAE ("Compute advantage and return", 330, 380-381; reading A3):
//   delta_t = r_t + disc_t V_{t+1} - V_t;  A_t = delta_t + disc_t lambda A_{t+1}, A_T = 0;  R_t = A_t + V_t
void gae(int T, int B, const double* V, const double* r, const uint8_t* d, double gamma, double lam,
         double* adv, double* ret) {
  for (int b = 0; b < B; ++b) {
    double a = 0.0;
    for (int t = T - 1; t >= 0; --t) {
      size_t i = (size_t)t * B + b;
      double disc = gamma * (1.0 - (double)d[i]);
      double delta = r[i] + disc * V[i + B] - V[i];
      a = delta + disc * lam * a;
      adv[i] = a; ret[i] = a + V[i];
    }
  }
}

// ---------------------------------------------------------------------------------------------
// O5 IMPALA actor-critic loss (coefficients PAPER.md:404-405; form = reading A4/A5/A6):
//   L = L_pg + c1 L_v + c2 L_ent,  L_pg = -mean pgadv log pi(a),  L_v = 1/2 mean (vs - V)^2,
//   L_ent = -mean H.   Seeds: dL/dl_i = (1/N)[-pgadv (1[i=a] - p_i) + c2 p_i (log p_i + H)],
//   dL/dV = -c1 (vs - V)/N.   "mean" becomes "sum" when reduction = 1.
// ---------------------------------------------------------------------------------------------
void impala_loss(int N, int A, const double* logits, const double* V, const int32_t* act,
                 const double* vs, const double* pgadv, const double* rho, double c1, double c2,
                 int reduction, double* stats, double* dlogits, double* dV) {
  double inv = reduction == 0 ? 1.0 / (double)N : 1.0;
  double s_pg = 0, s_v = 0, s_h = 0, s_rho = 0; vec lp(A);
  for (int n = 0; n < N; ++n) {
    log_softmax(logits + (size_t)n * A, A, lp.data());
    double H = entropy_of(lp.data(), A);
    double err = vs[n] - V[n];
    s_pg += -pgadv[n] * lp[act[n]]; s_v += 0.5 * err * err; s_h += H; if (rho) s_rho += rho[n];
    if (dlogits) for (int i = 0; i < A; ++i) {
      double p = std::exp(lp[i]);
      dlogits[(size_t)n * A + i] = inv * (-pgadv[n] * ((i == act[n] ? 1.0 : 0.0) - p) + c2 * p * (lp[i] + H));
    }
    if (dV) dV[n] = -c1 * err * inv;
  }
  stats[1] = s_pg * inv; stats[2] = s_v * inv; stats[3] = s_h / (double)N;
  stats[0] = stats[1] + c1 * stats[2] - c2 * (s_h * inv);
  stats[4] = 0; stats[5] = 0; stats[6] = 0; stats[7] = s_rho / (double)N;
}

// O7 PPO loss on one minibatch (Eq. 2, Eq. 3, Alg. 1 l.15-17
// PAPER.md:306-310, "Value Function Loss Clipping: False" PAPER.md:388; readings A5-A8):
//   Atil = (A - mean)/(std + 1e-8) (population std, two-pass);  r = exp(log pi(a) - logp_old)
//   L_pg = mean max(-Atil r, -Atil clip(r, 1-eps, 1+eps));  L_v = 1/2 mean (V - R)^2
//   L = L_pg + c1 L_v - c2 mean H;  approx_kl = mean((r-1) - log r);  clip_frac = mean(|r-1| > eps)
void ppo_loss(int m, int A, const double* logits, const double* V, const int32_t* act, const double* adv,
              const double* ret, const double* logp_old, double eps, double c1, double c2, int norm_adv,
              double* stats, double* dlogits, double* dV) {
  double mean = 0, var = 0;
  if (norm_adv) {
    for (int n = 0; n < m; ++n) mean += adv[n]; mean /= (double)m;
    for (int n = 0; n < m; ++n) var += (adv[n] - mean) * (adv[n] - mean); var /= (double)m;
  }
  double sd = std::sqrt(var), inv = 1.0 / (double)m;
  double s_pg = 0, s_v = 0, s_h = 0, s_kl = 0, s_cf = 0; vec lp(A);
  for (int n = 0; n < m; ++n) {
    log_softmax(logits + (size_t)n * A, A, lp.data());
    double H = entropy_of(lp.data(), A);
    double At = norm_adv ? (adv[n] - mean) / (sd + 1e-8) : adv[n];
    double logr = lp[act[n]] - logp_old[n], r = std::exp(logr);
    double rc = std::min(std::max(r, 1.0 - eps), 1.0 + eps);
    double l1 = -At * r, l2 = -At * rc;
    s_pg += std::max(l1, l2);
    // gradient flows through the unclipped branch unless strictly clipped on the penalised side (A7)
    bool clipped = (At > 0 && r > 1.0 + eps) || (At < 0 && r < 1.0 - eps);
    double dlogp = clipped ? 0.0 : -At * r * inv;
    double err = V[n] - ret[n];
    s_v += 0.5 * err * err; s_h += H; s_kl += (r - 1.0) - logr; s_cf += std::fabs(r - 1.0) > eps ? 1.0 : 0.0;
    if (dlogits) for (int i = 0; i < A; ++i) {
      double p = std::exp(lp[i]);
      dlogits[(size_t)n * A + i] = dlogp * ((i == act[n] ? 1.0 : 0.0) - p) + inv * c2 * p * (lp[i] + H);
    }
    if (dV) dV[n] = c1 * err * inv;
  }
  stats[1] = s_pg * inv; stats[2] = s_v * inv; stats[3] = s_h * inv;
  stats[0] = stats[1] + c1 * stats[2] - c2 * stats[3];
  stats[4] = 0; stats[5] = s_kl * inv; stats[6] = s_cf * inv; stats[7] = 0;
}

// O9 clip + Adam (Alg. 1 l.19-20 PAPER.md:313-315; Adam eps PAPER.md:389; readings A12, A13):
//   n = sqrt(sum g^2);  g <- g c / max(n, c);  m <- b1 m + (1-b1) g;  v <- b2 v + (1-b2) g^2
//   theta <- theta - lr (m/(1-b1^k)) / (sqrt(v/(1-b2^k)) + eps),  k = update count from 1.
double clip_adam(size_t P, float* theta, float* m, float* v, const double* g, uint64_t k, double lr,
                 double b1, double b2, double eps, double max_norm) {
  double ss = 0.0; for (size_t i = 0; i < P; ++i) ss += g[i] * g[i];
  double n = std::sqrt(ss), scale = max_norm / std::max(n, max_norm);
  double bc1 = 1.0 - std::pow(b1, (double)k), bc2 = 1.0 - std::pow(b2, (double)k);
  for (size_t i = 0; i < P; ++i) {
    double gi = g[i] * scale;
    double mi = b1 * (double)m[i] + (1.0 - b1) * gi;
    double vi = b2 * (double)v[i] + (1.0 - b2) * gi * gi;
    double th = (double)theta[i] - lr * (mi / bc1) / (std::sqrt(vi / bc2) + eps);
    m[i] = (float)mi; v[i] = (float)vi; theta[i] = (float)th;
  }
  return n;
}

// Reading A22, RMSprop as the paper's IMPALA optimizer (Table 3: "RMSprop eps 0.01, decay 0.99"; the
// paper's stack is optax): nu <- decay nu + (1-decay) g^2;  theta <- theta - lr g / sqrt(nu + eps)   (eps INSIDE the root,
// nu_0 = 0, no momentum, no centering), after the same global-norm clip as O9.  nu lives in the adam_v buffer.
double clip_rmsprop(size_t P, float* theta, float* nu, const double* g, double lr, double decay, double eps, double max_norm) {
  double ss = 0.0; for (size_t i = 0; i < P; ++i) ss += g[i] * g[i];
  double n = std::sqrt(ss), scale = max_norm / std::max(n, max_norm);
  for (size_t i = 0; i < P; ++i) {
    double gi = g[i] * scale;
    double ni = decay * (double)nu[i] + (1.0 - decay) * gi * gi;
    double th = (double)theta[i] - lr * gi / std::sqrt(ni + eps);
    nu[i] = (float)ni; theta[i] = (float)th;
  }
  return n;
}

// forward over F frames -> double logits [F,A], values [F]
void forward_many(const orc_arch& a, const Layout& L, const double* P, const uint8_t* obs, int F,
                  double* logits, double* values) {
  size_t fs = (size_t)a.in_c * a.in_h * a.in_w;
  for (int f = 0; f < F; ++f) net_forward(a, L, P, obs + fs * f, logits + (size_t)f * a.n_actions, values + f, nullptr);
}
// sum over frames of the per-frame adjoint (tape recomputed per frame to bound memory)
void backward_many(const orc_arch& a, const Layout& L, const double* P, const uint8_t* obs, const int32_t* frame_idx,
                   int F, const double* dlogits, const double* dV, double* G) {
  size_t fs = (size_t)a.in_c * a.in_h * a.in_w; Tape t; vec lg(a.n_actions); double val;
  for (int f = 0; f < F; ++f) {
    size_t src = frame_idx ? (size_t)frame_idx[f] : (size_t)f;
    net_forward(a, L, P, obs + fs * src, lg.data(), &val, &t);
    net_backward(a, L, P, t, dlogits + (size_t)f * a.n_actions, dV[f], G);
  }
}

}  // namespace

// =============================================================================================
// C entry points (ctypes).  All pointers are HOST pointers.
// =============================================================================================
extern "C" {

size_t orc_param_count(const orc_arch* a) { return make_layout(*a).total; }

// tensor i of the canonical parameter order: offset and element count; returns 0 past the end.
int orc_param_tensor(const orc_arch* a, int i, size_t* offset, size_t* count, int* fan_in) {
  Layout L = make_layout(*a); int nc = (int)L.convs.size();
  if (i < 2 * nc) { int li = i / 2; const LayerSpec& s = L.convs[li];
    if (i % 2 == 0) { *offset = L.conv_w[li]; *count = (size_t)s.cout * s.cin * s.k * s.k; } else { *offset = L.conv_b[li]; *count = s.cout; }
    *fan_in = s.cin * s.k * s.k; return 1; }
  i -= 2 * nc;
  size_t offs[6] = {L.fc_w, L.fc_b, L.pi_w, L.pi_b, L.v_w, L.v_b};
  size_t cnts[6] = {(size_t)a->fc * L.fc_in, (size_t)a->fc, (size_t)a->n_actions * a->fc, (size_t)a->n_actions, (size_t)a->fc, 1};
  int fans[6] = {L.fc_in, L.fc_in, a->fc, a->fc, a->fc, a->fc};
  if (i >= 6) return 0;
  *offset = offs[i]; *count = cnts[i]; *fan_in = fans[i]; return 1;
}

void orc_feature_shape(const orc_arch* a, int* c, int* h, int* w) { Layout L = make_layout(*a); *c = L.feat_c; *h = L.feat_h; *w = L.feat_w; }

// O1 forward, fp32 params in, fp64 out (logits64/values64) and/or fp32 out (ABI rounding point).
void orc_forward(const orc_arch* a, const float* params, const uint8_t* obs, int F,
                 double* logits64, double* values64, float* logits32, float* values32) {
  Layout L = make_layout(*a); vec P(params, params + L.total);
  vec lg((size_t)F * a->n_actions), vl(F);
  forward_many(*a, L, P.data(), obs, F, lg.data(), vl.data());
  for (size_t i = 0; i < lg.size(); ++i) { if (logits64) logits64[i] = lg[i]; if (logits32) logits32[i] = (float)lg[i]; }
  for (int i = 0; i < F; ++i) { if (values64) values64[i] = vl[i]; if (values32) values32[i] = (float)vl[i]; }
}

// same with fp64 parameters (finite-difference tests perturb parameters below fp32 resolution)
void orc_forward_f64(const orc_arch* a, const double* params, const uint8_t* obs, int F, double* logits, double* values) {
  Layout L = make_layout(*a); forward_many(*a, L, params, obs, F, logits, values);
}

// O8: G += sum_f J_f^T (dlogits_f, dV_f); fp64 parameters and gradient.
void orc_backward_f64(const orc_arch* a, const double* params, const uint8_t* obs, int F,
                      const double* dlogits, const double* dV, double* grad) {
  Layout L = make_layout(*a); backward_many(*a, L, params, obs, nullptr, F, dlogits, dV, grad);
}

void orc_log_softmax(const double* logits, int F, int A, double* logp, double* entropy) {
  for (int f = 0; f < F; ++f) { log_softmax(logits + (size_t)f * A, A, logp + (size_t)f * A); if (entropy) entropy[f] = entropy_of(logp + (size_t)f * A, A); }
}

// max-pool 3x3 s2 XLA-SAME on a [C,H,W] map: y [C,ceil(H/2),ceil(W/2)], arg = flat input index (A10, A11)
void orc_maxpool_same(const double* x, int Cc, int H, int W, double* y, int32_t* arg) {
  vec xv(x, x + (size_t)Cc * H * W), yv; std::vector<int> av; pool_fwd(xv, Cc, H, W, yv, av);
  for (size_t i = 0; i < yv.size(); ++i) { y[i] = yv[i]; arg[i] = av[i]; }
}

void orc_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }
double orc_fixed_log(double x) { return fixed_log(x); }
float orc_gumbel_from_u32(uint32_t x) { return gumbel_from_u32(x); }
void orc_gumbel_table(uint32_t lo, uint32_t n, float* out) { for (uint32_t i = 0; i < n; ++i) out[i] = gumbel_from_u32((lo + i) << 8); }
void orc_fixed_log_u24(uint32_t lo, uint32_t n, double* out) { for (uint32_t i = 0; i < n; ++i) out[i] = fixed_log(((double)(lo + i) + 0.5) * 0x1p-24); }

// O3 sampling for B envs: actions[b] from logits[b,:], counter env = env_offset + b.
void orc_sample(const float* logits, int B, int A, uint64_t seed, uint64_t step, uint32_t env_offset, int32_t* actions) {
  for (int b = 0; b < B; ++b) actions[b] = sample_action(logits + (size_t)b * A, A, seed, step, env_offset + (uint32_t)b);
}

void orc_permutation(uint64_t seed, uint32_t epoch, int N, int32_t* perm) { permutation(seed, epoch, N, perm); }

void orc_vtrace(int T, int B, const double* V, const double* r, const uint8_t* d, const double* logpi, const double* logmu,
                double gamma, double lam, double rho_bar, double c_bar, double rho_pg_bar, double* vs, double* pgadv, double* rho) {
  vtrace(T, B, V, r, d, logpi, logmu, gamma, lam, rho_bar, c_bar, rho_pg_bar, vs, pgadv, rho);
}
void orc_gae(int T, int B, const double* V, const double* r, const uint8_t* d, double gamma, double lam, double* adv, double* ret) {
  gae(T, B, V, r, d, gamma, lam, adv, ret);
}
void orc_impala_loss(int N, int A, const double* logits, const double* V, const int32_t* act, const double* vs, const double* pgadv,
                     const double* rho, double c1, double c2, int reduction, double* stats, double* dlogits, double* dV) {
  impala_loss(N, A, logits, V, act, vs, pgadv, rho, c1, c2, reduction, stats, dlogits, dV);
}
void orc_ppo_loss(int m, int A, const double* logits, const double* V, const int32_t* act, const double* adv, const double* ret,
                  const double* logp_old, double eps, double c1, double c2, int norm_adv, double* stats, double* dlogits, double* dV) {
  ppo_loss(m, A, logits, V, act, adv, ret, logp_old, eps, c1, c2, norm_adv, stats, dlogits, dV);
}
double orc_clip_rmsprop(size_t P, float* theta, float* nu, const double* g, double lr, double decay, double eps, double max_norm) {
  return clip_rmsprop(P, theta, nu, g, lr, decay, eps, max_norm);
}
// linear decay of the learning rate to 0 over `total` updates (Tables 2-3 "Anneal lr: linear"): lr_k = lr0 (1 - k/total)
double orc_linear_lr(double lr0, uint64_t k, uint64_t total) { return total ? lr0 * (1.0 - (double)std::min(k, total) / (double)total) : lr0; }
double orc_clip_adam(size_t P, float* theta, float* m, float* v, const double* g, uint64_t k, double lr, double b1, double b2,
                     double eps, double max_norm) { return clip_adam(P, theta, m, v, g, k, lr, b1, b2, eps, max_norm); }

// IMPALA loss as a function of fp64 parameters with the targets held constant (for finite
// differences of the "targets are constants" reading, A4): targets are computed at params_tgt.
double orc_impala_objective_f64(const orc_arch* a, const orc_hparams* hp, const double* params, const double* params_tgt,
                                const uint8_t* obs, const int32_t* actions, const float* rewards, const uint8_t* dones,
                                const float* behaviour_logits, double* grad /*nullable*/) {
  Layout L = make_layout(*a); int T = hp->T, B = hp->B, N = T * B, A = a->n_actions, F = (T + 1) * B;
  vec lg((size_t)F * A), V(F), lgt((size_t)F * A), Vt(F);
  forward_many(*a, L, params, obs, F, lg.data(), V.data());
  forward_many(*a, L, params_tgt, obs, F, lgt.data(), Vt.data());
  vec logpi(N), logmu(N), r(N), lp(A), bl(A);
  for (int n = 0; n < N; ++n) {
    log_softmax(&lgt[(size_t)n * A], A, lp.data()); logpi[n] = lp[actions[n]];
    for (int i = 0; i < A; ++i) bl[i] = behaviour_logits[(size_t)n * A + i];
    log_softmax(bl.data(), A, lp.data()); logmu[n] = lp[actions[n]]; r[n] = rewards[n];
  }
  vec vs(N), pg(N), rho(N);
  vtrace(T, B, Vt.data(), r.data(), dones, logpi.data(), logmu.data(), hp->gamma, hp->lambda_, hp->rho_bar, hp->c_bar, hp->rho_pg_bar, vs.data(), pg.data(), rho.data());
  double st[ORC_N_STATS]; vec dl((size_t)N * A), dV(N);
  impala_loss(N, A, lg.data(), V.data(), actions, vs.data(), pg.data(), rho.data(), hp->vf_coef, hp->ent_coef, hp->loss_reduction, st, dl.data(), dV.data());
  if (grad) { std::fill(grad, grad + L.total, 0.0); backward_many(*a, L, params, obs, nullptr, N, dl.data(), dV.data(), grad); }
  return st[0];
}

// PPO minibatch loss as a function of fp64 parameters (adv/ret/logp_old given), for finite differences.
double orc_ppo_objective_f64(const orc_arch* a, const orc_hparams* hp, const double* params, const uint8_t* obs, int m,
                             const int32_t* actions, const double* adv, const double* ret, const double* logp_old, double* grad) {
  Layout L = make_layout(*a); int A = a->n_actions;
  vec lg((size_t)m * A), V(m); forward_many(*a, L, params, obs, m, lg.data(), V.data());
  double st[ORC_N_STATS]; vec dl((size_t)m * A), dV(m);
  ppo_loss(m, A, lg.data(), V.data(), actions, adv, ret, logp_old, hp->clip_eps, hp->vf_coef, hp->ent_coef, hp->norm_adv, st, dl.data(), dV.data());
  if (grad) { std::fill(grad, grad + L.total, 0.0); backward_many(*a, L, params, obs, nullptr, m, dl.data(), dV.data(), grad); }
  return st[0];
}

// ---------------------------------------------------------------------------------------------
// The learner step (call stack SURVEY.md section 3 (4); Alg. 1 l.11-20 PAPER.md:296-315).
// Updates params/adam_m/adam_v in place (fp32 storage after every gradient update), increments
// *opt_step per update, writes stats[n_updates, 8].  Optional debug outputs (nullable):
//   out_logits [F,A], out_values [F] from the first forward; out_t0 / out_t1 [T*B] = (vs, pgadv)
//   or (adv, ret); out_grad [P] = gradient of the LAST update before clipping.
// ---------------------------------------------------------------------------------------------
int orc_learner_step(const orc_arch* a, const orc_hparams* hp, float* params, float* adam_m, float* adam_v, uint64_t* opt_step,
                     const uint8_t* obs, const int32_t* actions, const float* rewards, const uint8_t* dones,
                     const float* behaviour_logits, const float* behaviour_values /*nullable, [T+1,B]*/, float* stats,
                     double* out_logits, double* out_values, double* out_t0, double* out_t1, double* out_grad) {
  Layout L = make_layout(*a); int T = hp->T, B = hp->B, N = T * B, A = a->n_actions, F = (T + 1) * B;
  size_t P = L.total; vec Pd(params, params + P);
  vec lg((size_t)F * A), V(F);
  // Reading A3b (Alg. 1 l.8-12): PPO may be handed the values the ACTOR computed at rollout time
  // (v_t stored with the transition, v_next for the bootstrap observation); GAE then uses them and the learner's
  // iteration-start forward is not needed.  NULL = recompute them here with the iteration-start parameters (A3).
  // IMPALA ignores them: V-trace is defined on the current learner parameters' values (O4).
  const bool given_values = behaviour_values && hp->algo == 1;
  if (given_values) { for (int f = 0; f < F; ++f) V[f] = (double)behaviour_values[f]; std::fill(lg.begin(), lg.end(), 0.0); }
  else forward_many(*a, L, Pd.data(), obs, F, lg.data(), V.data());
  if (out_logits) std::copy(lg.begin(), lg.end(), out_logits);
  if (out_values) std::copy(V.begin(), V.end(), out_values);
  vec logmu(N), r(N), lp(A), bl(A);
  for (int n = 0; n < N; ++n) {
    for (int i = 0; i < A; ++i) bl[i] = behaviour_logits[(size_t)n * A + i];
    log_softmax(bl.data(), A, lp.data()); logmu[n] = lp[actions[n]]; r[n] = rewards[n];
  }
  vec G(P);
  if (hp->algo == 0) {
    // Reading A21 ("IMPALA ... 4 gradient updates per rollout", 401): the rollout is split by ENVIRONMENT into
    // `minibatches` groups of B/mb whole trajectories; each group is one complete update (forward with the current parameters,
    // V-trace, loss averaged over its T*B/mb samples, backward, clip, optimizer), applied in group order.  mb = 1 is the
    // single full-batch step of BASELINE.json configs 0/2/4.
    int mb = hp->minibatches < 1 ? 1 : hp->minibatches; int Bm = B / mb, Nm = T * Bm, Fm = (T + 1) * Bm;
    size_t fs = (size_t)a->in_c * a->in_h * a->in_w;
    for (int k = 0; k < mb; ++k) {
      std::vector<int32_t> fidx(Fm), act_m(Nm); std::vector<uint8_t> d_m(Nm); vec r_m(Nm), lmu_m(Nm);
      for (int t = 0; t <= T; ++t) for (int b = 0; b < Bm; ++b) fidx[(size_t)t * Bm + b] = t * B + k * Bm + b;
      for (int t = 0; t < T; ++t) for (int b = 0; b < Bm; ++b) { size_t src = (size_t)t * B + k * Bm + b, dst = (size_t)t * Bm + b;
        act_m[dst] = actions[src]; d_m[dst] = dones[src]; r_m[dst] = r[src]; lmu_m[dst] = logmu[src]; }
      if (mb > 1 || k > 0) Pd.assign(params, params + P);
      vec lgm((size_t)Fm * A), Vm(Fm);
      if (mb == 1) { lgm = lg; Vm = V; }
      else for (int f = 0; f < Fm; ++f) net_forward(*a, L, Pd.data(), obs + fs * fidx[f], &lgm[(size_t)f * A], &Vm[f], nullptr);
      vec logpi(Nm), vs(Nm), pg(Nm), rho(Nm);
      for (int n = 0; n < Nm; ++n) { log_softmax(&lgm[(size_t)n * A], A, lp.data()); logpi[n] = lp[act_m[n]]; }
      vtrace(T, Bm, Vm.data(), r_m.data(), d_m.data(), logpi.data(), lmu_m.data(), hp->gamma, hp->lambda_, hp->rho_bar, hp->c_bar, hp->rho_pg_bar, vs.data(), pg.data(), rho.data());
      if (out_t0 && mb == 1) std::copy(vs.begin(), vs.end(), out_t0);
      if (out_t1 && mb == 1) std::copy(pg.begin(), pg.end(), out_t1);
      double st[ORC_N_STATS]; vec dl((size_t)Nm * A), dV(Nm);
      impala_loss(Nm, A, lgm.data(), Vm.data(), act_m.data(), vs.data(), pg.data(), rho.data(), hp->vf_coef, hp->ent_coef, hp->loss_reduction, st, dl.data(), dV.data());
      std::fill(G.begin(), G.end(), 0.0);
      backward_many(*a, L, Pd.data(), obs, fidx.data(), Nm, dl.data(), dV.data(), G.data());   // bootstrap frames get no gradient
      if (out_grad) std::copy(G.begin(), G.end(), out_grad);
      *opt_step += 1;
      if (hp->optimizer == 1) st[4] = clip_rmsprop(P, params, adam_v, G.data(), hp->lr, hp->rms_decay, hp->rms_eps, hp->max_grad_norm);
      else st[4] = clip_adam(P, params, adam_m, adam_v, G.data(), *opt_step, hp->lr, hp->beta1, hp->beta2, hp->adam_eps, hp->max_grad_norm);
      for (int i = 0; i < ORC_N_STATS; ++i) stats[(size_t)k * ORC_N_STATS + i] = (float)st[i];
    }
    return mb;
  }
  // PPO (Alg. 1 l.11-20)
  vec adv(N), ret(N);
  gae(T, B, V.data(), r.data(), dones, hp->gamma, hp->lambda_, adv.data(), ret.data());
  if (out_t0) std::copy(adv.begin(), adv.end(), out_t0);
  if (out_t1) std::copy(ret.begin(), ret.end(), out_t1);
  int nmb = hp->minibatches, m = N / nmb, upd = 0;
  std::vector<int32_t> perm(N), act_m(m); vec adv_m(m), ret_m(m), lpo_m(m), lgm((size_t)m * A), Vm(m), dl((size_t)m * A), dV(m);
  size_t fs = (size_t)a->in_c * a->in_h * a->in_w;
  // Reading A23: the permutation of epoch e of this call is keyed by the epoch counter (opt_step at entry / minibatches) + e,
  // so successive calls of a training run (opt_step advances by epochs * minibatches per call) never reuse a partition.
  const uint32_t epoch0 = (uint32_t)(*opt_step / (uint64_t)nmb);
  for (int e = 0; e < hp->epochs; ++e) {
    permutation(hp->perm_seed, epoch0 + (uint32_t)e, N, perm.data());
    for (int k = 0; k < nmb; ++k, ++upd) {
      const int32_t* idx = &perm[(size_t)k * m];
      for (int j = 0; j < m; ++j) { act_m[j] = actions[idx[j]]; adv_m[j] = adv[idx[j]]; ret_m[j] = ret[idx[j]]; lpo_m[j] = logmu[idx[j]]; }
      Pd.assign(params, params + P);
      for (int j = 0; j < m; ++j) net_forward(*a, L, Pd.data(), obs + fs * idx[j], &lgm[(size_t)j * A], &Vm[j], nullptr);
      double st[ORC_N_STATS];
      ppo_loss(m, A, lgm.data(), Vm.data(), act_m.data(), adv_m.data(), ret_m.data(), lpo_m.data(), hp->clip_eps, hp->vf_coef, hp->ent_coef, hp->norm_adv, st, dl.data(), dV.data());
      std::fill(G.begin(), G.end(), 0.0);
      backward_many(*a, L, Pd.data(), obs, idx, m, dl.data(), dV.data(), G.data());
      if (out_grad) std::copy(G.begin(), G.end(), out_grad);
      *opt_step += 1;
      if (hp->optimizer == 1) st[4] = clip_rmsprop(P, params, adam_v, G.data(), hp->lr, hp->rms_decay, hp->rms_eps, hp->max_grad_norm);
      else st[4] = clip_adam(P, params, adam_m, adam_v, G.data(), *opt_step, hp->lr, hp->beta1, hp->beta2, hp->adam_eps, hp->max_grad_norm);
      for (int i = 0; i < ORC_N_STATS; ++i) stats[(size_t)upd * ORC_N_STATS + i] = (float)st[i];
    }
  }
  return upd;
}

}  // extern "C"
