// C ABI of include/cleanba.h: layer program construction, workspaces, and the two call stacks
// (SURVEY.md section 3 (3) cb_policy_forward, (4) cb_learner_step).
#include "common.cuh"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>

namespace cb {

static thread_local char g_err[512] = "";
void set_error(const char* fmt, ...) { va_list ap; va_start(ap, fmt); vsnprintf(g_err, sizeof g_err, fmt, ap); va_end(ap); }
int cuda_fail(cudaError_t e, const char* what) { set_error("CUDA error %s at %s", cudaGetErrorString(e), what); return CB_ECUDA; }

size_t wgrad_partial_elems(const Geom& g, long long frames);   // net.cu

static inline int pool_out_h(int h) { return (h + 1) / 2; }
static inline int conv_out_h(int h, int k, int s, int p) { return (h + 2 * p - k) / s + 1; }

struct Builder {
  cb_net* net; size_t off = 0; int cur = -1; int H, W, C;
  int tensor(size_t per_frame, bool f32 = false, int esize = 0) { net->tensors.push_back({per_frame, f32, esize}); return (int)net->tensors.size() - 1; }
  void need(int buf, size_t elems) { if (buf >= 0) net->grad_elems[buf] = std::max(net->grad_elems[buf], elems); }
  void ptensor(const std::string& name, size_t o, std::vector<int> dims, int fan) {
    cb_net::PT t; t.name = name; t.off = o; t.rank = (int)dims.size(); t.fan_in = fan;
    for (int i = 0; i < 4; ++i) t.dims[i] = i < (int)dims.size() ? dims[i] : 1;
    net->ptensors.push_back(t);
  }
  // appends a conv-shaped layer reading tensor `in`; returns layer index
  int conv(const std::string& name, int in, int cout, int kh, int kw, int s, int p, bool relu_in, int skip) {
    Layer L; L.name = name;
    L.g = {H, W, C, conv_out_h(H, kh, s, p), conv_out_h(W, kw, s, p), cout, kh, kw, s, p};
    size_t nw = (size_t)cout * C * kh * kw;
    L.pm = {off, off + nw, 0, 0, cout};
    ptensor(name + ".w", off, {cout, C, kh, kw}, C * kh * kw); ptensor(name + ".b", off + nw, {cout}, C * kh * kw);
    off += nw + cout;
    L.in_t = in; L.skip_t = skip; L.relu_in = relu_in; L.gate_in = relu_in; L.relu_out = false; L.u8_in = in < 0; L.f32_out = false;
    L.out_t = tensor((size_t)L.g.Ho * L.g.Wo * cout);
    L.wf_off = L.wd_off = net->wf_total; net->wf_total += (nw + 7) / 8 * 8;
    L.bias_off = net->bias_total; net->bias_total += (cout + 3) / 4 * 4;
    net->layers.push_back(L);
    H = L.g.Ho; W = L.g.Wo; C = cout;
    int li = (int)net->layers.size() - 1;
    net->fwd.push_back({OP_CONV, li, in, L.out_t, 0, 0, 0, -1, -1, -1, -1});
    return li;
  }
  void wgrad(int li, int dy) { net->bwd.push_back({OP_WGRAD, li, -1, -1, 0, 0, 0, dy, -1, -1, -1}); }
  void dgrad(int li, int dy, int dx, int add) {
    const Layer& L = net->layers[li];
    net->bwd.push_back({OP_DGRAD, li, -1, -1, 0, 0, 0, dy, dx, L.gate_in ? L.in_t : -1, add});
    need(dx, (size_t)L.g.H * L.g.W * L.g.Cin); need(dy, (size_t)L.g.Ho * L.g.Wo * L.g.Cout);
  }
};

static int build_program(cb_net* net) {
  const cb_arch& a = net->arch;
  Builder b; b.net = net; b.H = a.in_h; b.W = a.in_w; b.C = a.in_c;
  for (int i = 0; i < G_COUNT; ++i) net->grad_elems[i] = 0;
  net->wf_total = net->bias_total = 0;
  std::vector<int> convs;       // layer ids in forward order
  struct Stage { int conv, c_t, idx_t, C, H, W, l[4]; }; std::vector<Stage> stages;
  if (a.kind == CB_ARCH_NATURE) {
    convs.push_back(b.conv("conv1", -1, a.channels[0], 8, 8, 4, 0, false, -1));
    convs.push_back(b.conv("conv2", net->layers[convs[0]].out_t, a.channels[1], 4, 4, 2, 0, true, -1));
    convs.push_back(b.conv("conv3", net->layers[convs[1]].out_t, a.channels[2], 3, 3, 1, 0, true, -1));
    b.cur = net->layers[convs[2]].out_t;
  } else {
    for (int s = 0; s < 3; ++s) {
      char nm[64]; snprintf(nm, sizeof nm, "stage%d.conv", s);
      Stage st; st.conv = b.conv(nm, b.cur, a.channels[s], 3, 3, 1, 1, false, -1);
      st.c_t = net->layers[st.conv].out_t; st.C = b.C; st.H = b.H; st.W = b.W;
      int p = b.tensor((size_t)pool_out_h(b.H) * pool_out_h(b.W) * b.C);
      st.idx_t = b.tensor((size_t)pool_out_h(b.H) * pool_out_h(b.W) * b.C, false, 1);   // window position of the first maximum (A11)
      net->fwd.push_back({OP_POOL, -1, st.c_t, p, b.C, b.H, b.W, -1, -1, st.idx_t, -1});
      b.H = pool_out_h(b.H); b.W = pool_out_h(b.W);
      for (int k = 0; k < 2; ++k) {
        snprintf(nm, sizeof nm, "stage%d.block%d.conv1", s, k);
        st.l[2 * k] = b.conv(nm, p, a.channels[s], 3, 3, 1, 1, true, -1);
        snprintf(nm, sizeof nm, "stage%d.block%d.conv2", s, k);
        st.l[2 * k + 1] = b.conv(nm, net->layers[st.l[2 * k]].out_t, a.channels[s], 3, 3, 1, 1, true, p);
        // h = conv1(relu(p)) is only ever consumed as relu(h): conv1 stores relu(h), conv2 loads it as is
        net->layers[st.l[2 * k]].relu_out = true; net->layers[st.l[2 * k + 1]].relu_in = false;
        p = net->layers[st.l[2 * k + 1]].out_t;
      }
      b.cur = p; stages.push_back(st);
    }
  }
  if (b.H < 1 || b.W < 1) { set_error("input too small for this architecture"); return CB_EINVAL; }
  // the feature map is only ever consumed through a ReLU (by fc; its sign gates fc's dgrad all the same): the last conv stores relu(output)
  // and fc loads it as is
  net->layers.back().relu_out = true;
  int fc = b.conv("fc", b.cur, a.fc, b.H, b.W, 1, 0, false, -1);
  net->layers[fc].gate_in = true;
  net->hid_t = net->layers[fc].out_t;
  {  // the ABI reports fc.w as [out, in] with `in` flattened (C,H,W)
    cb_net::PT& t = net->ptensors[net->ptensors.size() - 2];
    t.rank = 2; t.dims[1] = t.dims[1] * t.dims[2] * t.dims[3]; t.dims[2] = t.dims[3] = 1;
  }
  // heads: 1x1 conv with A+1 outputs whose parameters are pi.w, pi.b, v.w, v.b in canonical order
  {
    int A = a.n_actions; size_t o = b.off;
    Layer L; L.name = "heads"; L.g = {1, 1, a.fc, 1, 1, A + 1, 1, 1, 1, 0};
    L.pm = {o, o + (size_t)A * a.fc, o + (size_t)A * a.fc + A, o + (size_t)A * a.fc + A + a.fc, A};
    b.ptensor("pi.w", L.pm.w_off, {A, a.fc}, a.fc); b.ptensor("pi.b", L.pm.b_off, {A}, a.fc);
    b.ptensor("v.w", L.pm.w2_off, {1, a.fc}, a.fc); b.ptensor("v.b", L.pm.b2_off, {1}, a.fc);
    b.off = L.pm.b2_off + 1;
    L.in_t = net->hid_t; L.skip_t = -1; L.relu_in = true; L.gate_in = true; L.relu_out = false; L.u8_in = false; L.f32_out = true;
    L.out_t = b.tensor((size_t)A + 1, true);
    size_t nw = (size_t)(A + 1) * a.fc;
    L.wf_off = L.wd_off = net->wf_total; net->wf_total += (nw + 7) / 8 * 8;
    L.bias_off = net->bias_total; net->bias_total += (A + 1 + 3) / 4 * 4;
    net->layers.push_back(L);
    net->fwd.push_back({OP_CONV, (int)net->layers.size() - 1, net->hid_t, L.out_t, 0, 0, 0, -1, -1, -1, -1});
    net->head_t = L.out_t;
  }
  net->wd_total = net->wf_total;
  net->P = b.off;
  // backward program; G_A carries the running gradient
  int heads = (int)net->layers.size() - 1;
  b.need(G_HEAD, (size_t)a.n_actions + 1);
  b.wgrad(heads, G_HEAD); b.dgrad(heads, G_HEAD, G_HID, -1);
  b.wgrad(fc, G_HID); b.dgrad(fc, G_HID, G_A, -1);
  if (a.kind == CB_ARCH_NATURE) {
    b.wgrad(convs[2], G_A); b.dgrad(convs[2], G_A, G_B, -1);
    b.wgrad(convs[1], G_B); b.dgrad(convs[1], G_B, G_A, -1);
    b.wgrad(convs[0], G_A);
  } else {
    for (int s = 2; s >= 0; --s) {
      const Stage& st = stages[s];
      for (int k = 1; k >= 0; --k) {
        int l1 = st.l[2 * k], l2 = st.l[2 * k + 1];
        b.wgrad(l2, G_A); b.dgrad(l2, G_A, G_B, -1);         // d(relu(h)) masked by h > 0
        b.wgrad(l1, G_B); b.dgrad(l1, G_B, G_A, G_A);        // block path + identity path (in place)
      }
      net->bwd.push_back({OP_POOLBWD, -1, st.c_t, -1, st.C, st.H, st.W, G_A, G_C, st.idx_t, -1});
      b.need(G_C, (size_t)st.C * st.H * st.W);
      b.wgrad(st.conv, G_C);
      if (s > 0) b.dgrad(st.conv, G_C, G_A, -1);
    }
  }
  return CB_OK;
}

static void drop_fwd_graphs(cb_net* net) {
  for (auto& fg : net->fwd_graphs) if (fg.exec) cudaGraphExecDestroy(fg.exec);
  net->fwd_graphs.clear();
}
static void free_workspace(Workspace& ws) {
  for (void* p : ws.act) cudaFree(p);
  ws.act.clear();
  for (int i = 0; i < G_COUNT; ++i) { cudaFree(ws.grad[i]); ws.grad[i] = nullptr; }
  cudaFree(ws.partial); ws.partial = nullptr; ws.frames = 0;
  cudaFree(ws.partial_tc); ws.partial_tc = nullptr; ws.partial_tc_elems = 0;
}
static void free_scratch(Workspace& ws) {
  void* ps[] = {ws.logpi, ws.logmu, ws.ent, ws.t0, ws.t1, ws.rho, ws.values, ws.terms, ws.red, ws.advstat, ws.perm, ws.permj, ws.act_m, ws.rew_m, ws.dones_m, ws.logmu_m};
  for (void* p : ps) cudaFree(p);
  ws.logpi = ws.logmu = ws.ent = ws.t0 = ws.t1 = ws.rho = ws.values = ws.terms = ws.advstat = nullptr; ws.red = nullptr; ws.perm = nullptr; ws.permj = nullptr;
  ws.act_m = nullptr; ws.rew_m = nullptr; ws.dones_m = nullptr; ws.logmu_m = nullptr;
  ws.learn_frames = ws.learn_N = ws.learn_epochs = 0;
}

#define CB_ALLOC(ptr, bytes) do { cudaError_t e__ = cudaMalloc((void**)&(ptr), (bytes) ? (bytes) : 16); if (e__ != cudaSuccess) { set_error("cudaMalloc of %zu bytes failed: %s", (size_t)(bytes), cudaGetErrorString(e__)); return CB_ENOMEM; } } while (0)

int ensure_workspace(cb_net* net, int prec, int frames) {
  Workspace& ws = net->ws[prec];
  size_t es = prec == CB_PREC_FP32_REF ? 4 : 2;
  if (!ws.wf) {
    CB_ALLOC(ws.wf, net->wf_total * es); CB_ALLOC(ws.wd, net->wd_total * es); CB_ALLOC(ws.bias, net->bias_total * 4);
    if (prec == CB_PREC_BF16_TC) { CB_ALLOC(ws.w0img, conv0_wimg_elems(net->layers[0].g) * 2); CB_ALLOC(ws.wtc_f, net->wf_total * 2); CB_ALLOC(ws.wtc_d, net->wf_total * 2); }
    CB_ALLOC(ws.errflag, 16); CB_CUDA(cudaMemset(ws.errflag, 0, 16));
    CB_CUDA(cudaHostAlloc((void**)&ws.errhost, 16, cudaHostAllocMapped)); *ws.errhost = 0;      // with UVA the host address is valid on the device
    {
      std::vector<PackDesc> tab;
      for (const Layer& L : net->layers)
        tab.push_back({L.g, L.pm, L.wf_off, L.bias_off, (prec == CB_PREC_BF16_TC && conv_tc_supported(L.g)) ? 1 : 0,
                       (prec == CB_PREC_BF16_TC && L.u8_in && conv0_tc_supported(L.g)) ? 1 : 0,
                       (prec == CB_PREC_BF16_TC && !L.u8_in && !L.f32_out && !L.relu_in && dense_tc_supported(L.g)) ? 1 : 0});
      CB_ALLOC(ws.packtab, tab.size() * sizeof(PackDesc));
      CB_CUDA(cudaMemcpy(ws.packtab, tab.data(), tab.size() * sizeof(PackDesc), cudaMemcpyHostToDevice));
    }
    CB_ALLOC(ws.gradbuf, net->P * 4); CB_ALLOC(ws.adam_scratch, clip_adam_scratch_bytes(net->P)); CB_ALLOC(ws.gnorm, 16);
  }
  if (ws.frames >= frames) return CB_OK;
  frames = std::max(frames, net->max_frames);
  CB_CUDA(cudaDeviceSynchronize());
  drop_fwd_graphs(net);      // they hold the old activation pointers
  free_workspace(ws);
  ws.act.assign(net->tensors.size(), nullptr);
  for (size_t i = 0; i < net->tensors.size(); ++i)
    CB_ALLOC(ws.act[i], net->tensors[i].per_frame * frames * (net->tensors[i].esize ? (size_t)net->tensors[i].esize : (net->tensors[i].f32 ? 4 : es)));
  for (int i = 0; i < G_COUNT; ++i) CB_ALLOC(ws.grad[i], net->grad_elems[i] * frames * es);
  size_t pe = 0;
  for (const Layer& L : net->layers) {
    pe = std::max(pe, wgrad_partial_elems(L.g, frames));
    if (wgrad_tc_supported(L.g)) pe = std::max(pe, wgrad_tc_partial_elems(L.g));
    if (L.u8_in && conv0_tc_supported(L.g)) pe = std::max(pe, conv0_partial_elems(L.g));
    if (dense_tc_supported(L.g)) pe = std::max(pe, dense_partial_elems(L.g, frames));
  }
  CB_ALLOC(ws.partial, pe * 4); ws.partial_elems = pe;
  if (prec == CB_PREC_BF16_TC) {
    size_t pt = 0;
    for (const Layer& L : net->layers) if (wgrad_tc_supported(L.g)) pt += wgrad_tc_partial_elems(L.g);
    if (pt) { CB_ALLOC(ws.partial_tc, pt * 4); ws.partial_tc_elems = pt; }
  }
  ws.frames = frames;
  return CB_OK;
}

int ensure_learner_scratch(cb_net* net, int prec, int F, int N, int epochs) {
  Workspace& ws = net->ws[prec];
  if (ws.learn_frames >= F && ws.learn_N >= N && ws.learn_epochs >= epochs) return CB_OK;
  F = std::max(F, ws.learn_frames); N = std::max(N, ws.learn_N); epochs = std::max(std::max(epochs, 1), ws.learn_epochs);      // grow-only: take the maxima BEFORE the old sizes are cleared
  CB_CUDA(cudaDeviceSynchronize());
  free_scratch(ws);
  size_t n4 = (size_t)N * 4;
  CB_ALLOC(ws.logpi, n4); CB_ALLOC(ws.logmu, n4); CB_ALLOC(ws.ent, n4); CB_ALLOC(ws.t0, n4); CB_ALLOC(ws.t1, n4); CB_ALLOC(ws.rho, n4);
  CB_ALLOC(ws.values, (size_t)F * (net->arch.n_actions + 1) * 4);
  CB_ALLOC(ws.terms, 16); CB_ALLOC(ws.red, 256 + (size_t)((N + 127) / 128) * 40); CB_ALLOC(ws.advstat, 16);      // red: [0..1] advantage mean / std, [8..] per-block loss-term partials
  CB_ALLOC(ws.perm, std::max(n4 * epochs, (size_t)F * 4)); CB_ALLOC(ws.permj, n4 * epochs);
  CB_ALLOC(ws.act_m, n4); CB_ALLOC(ws.rew_m, n4); CB_ALLOC(ws.dones_m, (size_t)N); CB_ALLOC(ws.logmu_m, n4);
  ws.learn_frames = F; ws.learn_N = N; ws.learn_epochs = epochs;
  return CB_OK;
}

// Philox4x32-10 on the host, for cb_net_init only (A14)
static void philox_host(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t out[4]) {
  for (int r = 0; r < 10; ++r) {
    uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    c0 = n0; c1 = (uint32_t)p1; c2 = n2; c3 = (uint32_t)p0; k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// one opt-in per (device, kernel); the cache is guarded: cb_net objects of different host threads share it
int ensure_dyn_smem(const void* func, size_t bytes) {
  static std::mutex mu; static std::map<std::pair<int, const void*>, size_t> done;
  int dev = 0; CB_CUDA(cudaGetDevice(&dev));
  std::lock_guard<std::mutex> lk(mu);
  size_t& cur = done[{dev, func}];
  if (bytes <= cur) return CB_OK;
  CB_CUDA(cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
  cur = bytes;
  return CB_OK;
}

}  // namespace cb

using namespace cb;

extern "C" {

const char* cb_last_error(void) { return g_err; }

int cb_net_create(const cb_arch* arch, int max_frames, cb_net** out) {
  if (out) *out = nullptr;
  if (!arch || !out) { set_error("null argument"); return CB_EINVAL; }
  if ((arch->kind != CB_ARCH_NATURE && arch->kind != CB_ARCH_IMPALA) || arch->in_c < 1 || arch->in_h < 1 || arch->in_w < 1 || arch->fc < 1 ||
      arch->n_actions < 1 || arch->n_actions > 31 || arch->channels[0] < 1 || arch->channels[1] < 1 || arch->channels[2] < 1) {
    set_error("bad architecture description"); return CB_EINVAL;
  }
  if (arch->kind == CB_ARCH_NATURE && (arch->in_h < 36 || arch->in_w < 36)) { set_error("Nature-CNN needs an input of at least 36x36"); return CB_EINVAL; }
  cb_net* net = new (std::nothrow) cb_net();
  if (!net) { set_error("out of host memory"); return CB_ENOMEM; }
  net->arch = *arch; net->max_frames = std::max(max_frames, 0);
  int rc = build_program(net);
  if (rc) { delete net; return rc; }
  *out = net;
  return CB_OK;
}

void cb_net_destroy(cb_net* net) {
  if (!net) return;
  cudaDeviceSynchronize();
  drop_fwd_graphs(net);
  if (net->capture_stream) cudaStreamDestroy(net->capture_stream);
  if (net->aux_stream) { cudaStreamDestroy(net->aux_stream); cudaEventDestroy(net->ev_fork); cudaEventDestroy(net->ev_join); }
  for (int p = 0; p < 2; ++p) {
    Workspace& ws = net->ws[p];
    if (!ws.wf) continue;
    free_workspace(ws); free_scratch(ws);
    cudaFree(ws.packtab); cudaFree(ws.w0img); cudaFree(ws.wtc_f); cudaFree(ws.wtc_d); cudaFree(ws.errflag); cudaFreeHost(ws.errhost);
    cudaFree(ws.wf); cudaFree(ws.wd); cudaFree(ws.bias); cudaFree(ws.gradbuf); cudaFree(ws.adam_scratch); cudaFree(ws.gnorm);
  }
  delete net;
}

size_t cb_param_count(const cb_net* net) { return net ? net->P : 0; }

int cb_param_layout(const cb_net* net, int i, const char** name, size_t* offset, int* rank, int dims[4]) {
  if (!net || i < 0 || i >= (int)net->ptensors.size()) { set_error("tensor index out of range"); return CB_EINVAL; }
  const cb_net::PT& t = net->ptensors[i];
  if (name) *name = t.name.c_str();
  if (offset) *offset = t.off;
  if (rank) *rank = t.rank;
  if (dims) for (int k = 0; k < 4; ++k) dims[k] = t.dims[k];
  return CB_OK;
}

int cb_net_init(const cb_net* net, uint64_t seed, float* params_host) {
  if (!net || !params_host) { set_error("null argument"); return CB_EINVAL; }
  const double TWO_PI = 6.283185307179586476925286766559;
  for (size_t ti = 0; ti < net->ptensors.size(); ++ti) {
    const cb_net::PT& t = net->ptensors[ti];
    size_t n = 1; for (int k = 0; k < t.rank; ++k) n *= (size_t)t.dims[k];
    bool is_w = t.name.size() >= 2 && t.name.compare(t.name.size() - 2, 2, ".w") == 0;
    if (!is_w) { for (size_t i = 0; i < n; ++i) params_host[t.off + i] = 0.f; continue; }
    double sd = std::sqrt(2.0 / (double)t.fan_in);
    for (size_t j = 0; j * 4 < n; ++j) {
      uint32_t r[4]; philox_host((uint32_t)j, (uint32_t)(j >> 32), (uint32_t)ti, 0x494E4954u, (uint32_t)seed, (uint32_t)(seed >> 32), r);
      for (int h = 0; h < 2; ++h) {
        double u1 = ((double)(r[2 * h] >> 8) + 0.5) * 0x1p-24, u2 = ((double)(r[2 * h + 1] >> 8) + 0.5) * 0x1p-24;
        double rad = std::sqrt(-2.0 * std::log(u1));
        double z[2] = {rad * std::cos(TWO_PI * u2), rad * std::sin(TWO_PI * u2)};
        for (int q = 0; q < 2; ++q) { size_t i = j * 4 + 2 * h + q; if (i < n) params_host[t.off + i] = (float)(sd * z[q]); }
      }
    }
  }
  return CB_OK;
}

static int check_prec(int prec) { if (prec != CB_PREC_FP32_REF && prec != CB_PREC_BF16_TC) { set_error("bad precision mode"); return CB_EINVAL; } return CB_OK; }
static bool misaligned(const void* p, size_t a) { return ((uintptr_t)p & (a - 1)) != 0; }

// raised host word -> CB_ECUDA once, condition cleared (cleanba.h, asynchronous errors)
static int report_async_error(cb_net* net, cudaStream_t st) {
  int code = 0;
  for (int p = 0; p < 2; ++p) {
    Workspace& ws = net->ws[p];
    if (!ws.errhost) continue;
    const int h = *(volatile int*)ws.errhost;
    if (h) { code = h; *(volatile int*)ws.errhost = 0; cudaMemsetAsync(ws.errflag, 0, sizeof(int), st); ws.packed = false; }
  }
  if (!code) return CB_OK;
  set_error("a tcgen05 pipeline wait timed out inside an earlier call on this net (site %d): that call's stats / logits were poisoned with NaN and its optimizer step was skipped", code);
  return CB_ECUDA;
}

// The actor calls the trunk thousands of times with the same shapes and a handful of observation buffers, and at B = 128 its
// ~18 kernels are shorter than their host-side launch cost (tensor-map encoding included).  The first call with a given
// (precision, B, obs pointer) runs eagerly, the second is captured into a CUDA graph on a private stream, later ones replay it
// on the caller's stream.  Weights and activations live in library-owned buffers whose addresses only change in
// ensure_workspace, which drops the graphs.  Event-timed profiling (cb_profile_begin) uses the eager path.
static int trunk_forward(cb_net* net, int precision, const uint8_t* obs, int B, cudaStream_t st) {
  if (prof_active()) return forward(net, precision, obs, nullptr, B, st, true);
  cb_net::FwdGraph* fg = nullptr;
  for (auto& e : net->fwd_graphs) if (e.prec == precision && e.B == B && e.obs == obs) { fg = &e; break; }
  if (!fg) {
    if (net->fwd_graphs.size() >= 64) drop_fwd_graphs(net);
    net->fwd_graphs.push_back({precision, B, obs, nullptr, 0, false});
    return forward(net, precision, obs, nullptr, B, st, true);
  }
  if (fg->bad) return forward(net, precision, obs, nullptr, B, st, true);
  if (!fg->exec) {
    if (!net->capture_stream) CB_CUDA(cudaStreamCreateWithFlags(&net->capture_stream, cudaStreamNonBlocking));
    const uint64_t l0 = cb_launch_count();
    cudaGraph_t graph = nullptr;
    CB_CUDA(cudaStreamBeginCapture(net->capture_stream, cudaStreamCaptureModeRelaxed));
    const int rc = forward(net, precision, obs, nullptr, B, net->capture_stream, true);
    const cudaError_t ce = cudaStreamEndCapture(net->capture_stream, &graph);
    fg->launches = cb_launch_count() - l0;
    if (rc == CB_OK && ce == cudaSuccess && graph && cudaGraphInstantiate(&fg->exec, graph, 0) == cudaSuccess) {
      cudaGraphDestroy(graph);
      CB_CUDA(cudaGraphLaunch(fg->exec, st));
      return CB_OK;
    }
    if (graph) cudaGraphDestroy(graph);
    (void)cudaGetLastError();
    fg->exec = nullptr; fg->bad = true;      // not capturable here: stay eager (the counted launches of the failed capture are re-counted below)
    return forward(net, precision, obs, nullptr, B, st, true);
  }
  CB_CUDA(cudaGraphLaunch(fg->exec, st));
  prof_add_launches(fg->launches);
  return CB_OK;
}

int cb_policy_forward(cb_net* net, const float* params, const uint8_t* obs, int B, uint64_t seed, uint64_t step, uint32_t env_offset,
                      int precision, float* logits, float* value, int32_t* actions, void* stream) {
  if (!net || !obs || B < 0) { set_error("null or negative argument"); return CB_EINVAL; }
  if (check_prec(precision)) return CB_EINVAL;
  if (params && misaligned(params, 16)) { set_error("params must be 16-byte aligned"); return CB_EINVAL; }
  if (misaligned(obs, 4)) { set_error("obs must be 4-byte aligned"); return CB_EINVAL; }
  if (B == 0) return CB_OK;
  cudaStream_t st = (cudaStream_t)stream; int rc;
  if ((rc = report_async_error(net, st))) return rc;
  if ((rc = ensure_workspace(net, precision, B))) return rc;
  if (params) { if ((rc = pack_weights(net, precision, params, st))) return rc; }
  else if (!net->ws[precision].packed) { set_error("params == NULL but this net holds no current packed weights in this precision mode (none packed yet, or a learner call has run since)"); return CB_EINVAL; }
  if ((rc = trunk_forward(net, precision, obs, B, st))) return rc;      // everything up to the hidden layer
  Workspace& ws = net->ws[precision];
  const Layer& HL = net->layers.back();
  const int A = net->arch.n_actions;
  const size_t es = precision == CB_PREC_FP32_REF ? 4 : 2;
  if ((rc = launch_heads_sample(precision, ws.act[net->hid_t], (const char*)ws.wf + HL.wf_off * es, ws.bias + HL.bias_off, B, net->arch.fc, A, seed, step,
                                env_offset, (float*)ws.act[net->head_t], logits, value, actions, st, ws.errflag, ws.errhost))) return rc;
  return CB_OK;
}

// The operand-layout weights of an update: packed from the CURRENT master parameters at the start of every gradient computation.
static int learner_optimizer(cb_net* net, Workspace& ws, int u, cudaStream_t st) {
  cb_net::LearnCtx& c = net->lc; const cb_hparams& hp = c.hp;
  float* row = c.stats + (size_t)u * CB_N_STATS;
  *c.opt_step += 1;
  if (hp.optimizer == 1)
    return launch_clip_rmsprop(net->P, c.params, c.adam_v, ws.gradbuf, hp.lr, hp.rms_decay, hp.rms_eps, hp.max_grad_norm, ws.gnorm, row + 4, ws.adam_scratch, st, ws.errflag, ws.errhost);
  return launch_clip_adam(net->P, c.params, c.adam_m, c.adam_v, ws.gradbuf, *c.opt_step, hp.lr, hp.beta1, hp.beta2, hp.adam_eps, hp.max_grad_norm, ws.gnorm, row + 4,
                          ws.adam_scratch, st, ws.errflag, ws.errhost);
}

int cb_learner_begin(cb_net* net, float* params, float* adam_m, float* adam_v, uint64_t* opt_step, const uint8_t* obs, const int32_t* actions,
                     const float* rewards, const uint8_t* dones, const float* behaviour_logits, const float* behaviour_values, const cb_hparams* hp,
                     float* stats, void* stream) {
  if (!net || !params || !adam_m || !adam_v || !opt_step || !obs || !actions || !rewards || !dones || !behaviour_logits || !hp || !stats) { set_error("null argument"); return CB_EINVAL; }
  if (check_prec(hp->precision)) return CB_EINVAL;
  if (hp->algo != CB_ALGO_IMPALA && hp->algo != CB_ALGO_PPO) { set_error("bad algo"); return CB_EINVAL; }
  if (hp->T < 1 || hp->B < 1) { set_error("T and B must be positive"); return CB_EINVAL; }
  if (misaligned(params, 16) || misaligned(adam_m, 16) || misaligned(adam_v, 16)) { set_error("params / adam buffers must be 16-byte aligned"); return CB_EINVAL; }
  if (misaligned(obs, 4)) { set_error("obs must be 4-byte aligned"); return CB_EINVAL; }
  const int prec = hp->precision, T = hp->T, B = hp->B, A = net->arch.n_actions;
  if ((long long)(T + 1) * B * net->arch.in_h * net->arch.in_w >= 0x7fffffffLL) { set_error("(T+1)*B*H*W must stay below 2^31"); return CB_EINVAL; }
  const int N = T * B, F = (T + 1) * B;
  const bool ppo = hp->algo == CB_ALGO_PPO;
  if (ppo && (hp->epochs < 1 || hp->minibatches < 1 || N % hp->minibatches != 0)) { set_error("PPO needs epochs >= 1 and minibatches dividing T*B"); return CB_EINVAL; }
  const int mb = ppo ? hp->minibatches : (hp->minibatches < 1 ? 1 : hp->minibatches);
  if (!ppo && B % mb != 0) { set_error("IMPALA needs minibatches dividing B (env groups, A21)"); return CB_EINVAL; }
  if (hp->optimizer != 0 && hp->optimizer != 1) { set_error("bad optimizer"); return CB_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream; int rc;
  net->lc.active = false;
  if ((rc = report_async_error(net, st))) return rc;
  if ((rc = ensure_workspace(net, prec, F))) return rc;
  if ((rc = ensure_learner_scratch(net, prec, F, N, ppo ? hp->epochs : 1))) return rc;
  Workspace& ws = net->ws[prec];
  const bool given_values = ppo && behaviour_values;
  net->last_prec = prec; net->last_F = F; net->last_N = N; net->last_ppo = ppo || mb > 1; net->last_has_head = !given_values && (ppo || mb == 1);
  cb_net::LearnCtx& c = net->lc;
  c.params = params; c.adam_m = adam_m; c.adam_v = adam_v; c.opt_step = opt_step; c.obs = obs; c.actions = actions; c.rewards = rewards; c.dones = dones;
  c.stats = stats; c.hp = *hp; c.mb = mb; c.ppo = ppo; c.next_grad = c.next_apply = 0;
  c.n_updates = ppo ? hp->epochs * hp->minibatches : mb;
  // old log-probs log mu(a|s) from the behaviour logits (O4 / O6)
  if ((rc = launch_logprob(behaviour_logits, A, N, A, actions, nullptr, ws.logmu, nullptr, st))) return rc;
  float* head = (float*)ws.act[net->head_t];
  if (ppo) {
    // Alg. 1 l.11-12: advantages and returns, from the actor's values (A3b) or from a no-grad forward with the iteration-start
    // parameters (A3).  The epoch permutations (A17, A23) are independent of both: they run on a side stream underneath.
    if (!net->aux_stream) { CB_CUDA(cudaStreamCreateWithFlags(&net->aux_stream, cudaStreamNonBlocking)); CB_CUDA(cudaEventCreateWithFlags(&net->ev_fork, cudaEventDisableTiming)); CB_CUDA(cudaEventCreateWithFlags(&net->ev_join, cudaEventDisableTiming)); }
    CB_CUDA(cudaEventRecord(net->ev_fork, st)); CB_CUDA(cudaStreamWaitEvent(net->aux_stream, net->ev_fork, 0));
    if ((rc = launch_permutation(hp->perm_seed, (uint32_t)(*opt_step / (uint64_t)hp->minibatches), hp->epochs, N, ws.perm, ws.permj, net->aux_stream))) return rc;
    CB_CUDA(cudaEventRecord(net->ev_join, net->aux_stream));
    if (given_values) {
      if ((rc = launch_gae(T, B, behaviour_values, 1, rewards, dones, hp->gamma, hp->lambda_, ws.t0, ws.t1, st))) return rc;
    } else {
      if ((rc = pack_weights(net, prec, params, st))) return rc;
      if ((rc = forward(net, prec, obs, nullptr, F, st))) return rc;
      CB_CUDA(cudaMemcpyAsync(ws.values, head, (size_t)F * (A + 1) * 4, cudaMemcpyDeviceToDevice, st));      // cb_learner_view(0)
      if ((rc = launch_gae(T, B, ws.values + A, A + 1, rewards, dones, hp->gamma, hp->lambda_, ws.t0, ws.t1, st))) return rc;
    }
    CB_CUDA(cudaStreamWaitEvent(st, net->ev_join, 0));
  }
  c.active = true;
  return c.n_updates;
}

int cb_learner_grad(cb_net* net, int u, float** grad_dev, void* stream) {
  if (!net || !net->lc.active) { set_error("cb_learner_grad without cb_learner_begin"); return CB_EINVAL; }
  cb_net::LearnCtx& c = net->lc; const cb_hparams& hp = c.hp;
  if (u != c.next_grad || u != c.next_apply || u >= c.n_updates) { set_error("updates must be taken in order, each cb_learner_grad followed by its cb_learner_apply"); return CB_EINVAL; }
  cudaStream_t st = (cudaStream_t)stream; int rc;
  const int prec = hp.precision, T = hp.T, B = hp.B, A = net->arch.n_actions, N = T * B, F = (T + 1) * B;
  Workspace& ws = net->ws[prec];
  float* head = (float*)ws.act[net->head_t];
  float* row = c.stats + (size_t)u * CB_N_STATS;
  if (!(c.ppo && u == 0 && net->last_has_head)) { if ((rc = pack_weights(net, prec, c.params, st))) return rc; }      // PPO update 0 after the no-grad forward: same parameters, already packed
  ws.packed = false;      // after this call the packs no longer hold what `params` holds (the optimizer runs next)
  if (!c.ppo && c.mb == 1) {
    if ((rc = forward(net, prec, c.obs, nullptr, F, st, false, c.actions, N, ws.logpi))) return rc;      // log pi(a_t) comes out of the heads kernel
    if ((rc = launch_vtrace(T, B, head + A, A + 1, c.rewards, c.dones, ws.logpi, ws.logmu, hp.gamma, hp.lambda_, hp.rho_bar, hp.c_bar, hp.rho_pg_bar, ws.t0, ws.t1, ws.rho, st))) return rc;
    if ((rc = launch_impala_loss(prec, N, A, head, c.actions, ws.t0, ws.t1, ws.rho, hp.vf_coef, hp.ent_coef, hp.loss_reduction, ws.grad[G_HEAD], ws.terms, ws.red, row, st))) return rc;
    if ((rc = backward(net, prec, c.obs, nullptr, N, ws.gradbuf, st))) return rc;
  } else if (!c.ppo) {
    // A21: one complete update per group of B/mb envs, in group order, each with the parameters the previous one left
    const int Bm = B / c.mb, Nm = T * Bm, Fm = (T + 1) * Bm;
    if ((rc = launch_gather_traj(T, B, u * Bm, Bm, c.actions, c.rewards, c.dones, ws.logmu, ws.perm, ws.act_m, ws.rew_m, ws.dones_m, ws.logmu_m, st))) return rc;
    if ((rc = forward(net, prec, c.obs, ws.perm, Fm, st, false, ws.act_m, Nm, ws.logpi))) return rc;
    if ((rc = launch_vtrace(T, Bm, head + A, A + 1, ws.rew_m, ws.dones_m, ws.logpi, ws.logmu_m, hp.gamma, hp.lambda_, hp.rho_bar, hp.c_bar, hp.rho_pg_bar, ws.t0, ws.t1, ws.rho, st))) return rc;
    if ((rc = launch_impala_loss(prec, Nm, A, head, ws.act_m, ws.t0, ws.t1, ws.rho, hp.vf_coef, hp.ent_coef, hp.loss_reduction, ws.grad[G_HEAD], ws.terms, ws.red, row, st))) return rc;
    if ((rc = backward(net, prec, c.obs, ws.perm, Nm, ws.gradbuf, st))) return rc;
  } else {
    const int m = N / hp.minibatches, e = u / hp.minibatches, k = u % hp.minibatches;
    const int32_t* idx = ws.perm + (size_t)e * N + (size_t)k * m;
    if ((rc = forward(net, prec, c.obs, idx, m, st))) return rc;
    if ((rc = launch_ppo_loss(prec, m, A, head, idx, c.actions, ws.t0, ws.t1, ws.logmu, hp.clip_eps, hp.vf_coef, hp.ent_coef, hp.norm_adv, ws.grad[G_HEAD], ws.terms, ws.red, ws.advstat, row, st))) return rc;
    if ((rc = backward(net, prec, c.obs, idx, m, ws.gradbuf, st))) return rc;
  }
  c.next_grad = u + 1;
  if (grad_dev) *grad_dev = ws.gradbuf;
  return CB_OK;
}

int cb_learner_apply(cb_net* net, int u, void* stream) {
  if (!net || !net->lc.active) { set_error("cb_learner_apply without cb_learner_begin"); return CB_EINVAL; }
  cb_net::LearnCtx& c = net->lc;
  if (u != c.next_apply || c.next_grad != u + 1) { set_error("cb_learner_apply(%d) must follow cb_learner_grad(%d)", u, u); return CB_EINVAL; }
  int rc = learner_optimizer(net, net->ws[c.hp.precision], u, (cudaStream_t)stream);
  if (rc) return rc;
  c.next_apply = u + 1;
  if (c.next_apply == c.n_updates) c.active = false;
  return CB_OK;
}

int cb_learner_step(cb_net* net, float* params, float* adam_m, float* adam_v, uint64_t* opt_step, const uint8_t* obs, const int32_t* actions,
                    const float* rewards, const uint8_t* dones, const float* behaviour_logits, const float* behaviour_values, const cb_hparams* hp,
                    float* stats, void* stream) {
  const int n = cb_learner_begin(net, params, adam_m, adam_v, opt_step, obs, actions, rewards, dones, behaviour_logits, behaviour_values, hp, stats, stream);
  if (n < 0) return n;
  for (int u = 0; u < n; ++u) {
    int rc;
    if ((rc = cb_learner_grad(net, u, nullptr, stream))) { net->lc.active = false; return rc; }
    if ((rc = cb_learner_apply(net, u, stream))) { net->lc.active = false; return rc; }
  }
  return n;
}

int cb_check_errors(cb_net* net, void* stream) {
  if (!net) { set_error("null argument"); return CB_EINVAL; }
  CB_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
  return report_async_error(net, (cudaStream_t)stream);
}

int cb_debug_inject_timeout(cb_net* net, int precision, void* stream) {
  if (!net || check_prec(precision)) return CB_EINVAL;
  Workspace& ws = net->ws[precision];
  if (!ws.errflag) { set_error("no workspace in this precision mode yet"); return CB_EINVAL; }
  const int one = 99;
  CB_CUDA(cudaMemcpyAsync(ws.errflag, &one, sizeof one, cudaMemcpyHostToDevice, (cudaStream_t)stream));
  return CB_OK;
}

int cb_sum_ranks(const float* in, int G, size_t n, float scale, float* out, void* stream) {
  if (!in || !out || G < 1) { set_error("bad argument"); return CB_EINVAL; }
  return launch_sum_ranks(in, G, n, scale, out, (cudaStream_t)stream);
}

int cb_learner_view(const cb_net* net, int which, const void** dev_ptr, size_t* count) {
  if (!net || !dev_ptr || !count || net->last_prec < 0) { set_error("no learner step has run on this net"); return CB_EINVAL; }
  const Workspace& ws = net->ws[net->last_prec]; int A = net->arch.n_actions;
  switch (which) {
    case 0: if (!net->last_has_head) { set_error("view 0: the last call ran no forward over all (T+1)B frames (PPO with behaviour_values, or IMPALA env groups)"); return CB_EINVAL; }
            *dev_ptr = net->last_ppo ? (const void*)ws.values : (const void*)ws.act[net->head_t]; *count = (size_t)net->last_F * (A + 1); break;
    case 1: *dev_ptr = ws.t0; *count = net->last_N; break;
    case 2: *dev_ptr = ws.t1; *count = net->last_N; break;
    case 3: *dev_ptr = ws.gradbuf; *count = net->P; break;
    default: set_error("bad view index"); return CB_EINVAL;
  }
  return CB_OK;
}

int cb_sample_actions(const float* logits, int B, int A, uint64_t seed, uint64_t step, uint32_t env_offset, int32_t* actions, void* stream) {
  if (!logits || !actions || B < 0 || A < 1) { set_error("bad argument"); return CB_EINVAL; }
  return launch_sample(logits, A, B, A, seed, step, env_offset, actions, (cudaStream_t)stream);
}
int cb_logprob_entropy(const float* logits, int ld, int N, int A, const int32_t* actions, float* logp_a, float* entropy, void* stream) {
  if (!logits || !actions || N < 0 || A < 1 || A > 32 || ld < A) { set_error("bad argument"); return CB_EINVAL; }
  return launch_logprob(logits, ld, N, A, actions, nullptr, logp_a, entropy, (cudaStream_t)stream);
}
int cb_vtrace(int T, int B, const float* V, const float* r, const uint8_t* d, const float* logpi, const float* logmu, float gamma, float lambda_,
              float rho_bar, float c_bar, float rho_pg_bar, float* vs, float* pgadv, float* rho, void* stream) {
  if (T < 0 || B < 0) { set_error("bad argument"); return CB_EINVAL; }
  if (T == 0 || B == 0) return CB_OK;
  if (!V || !r || !d || !logpi || !logmu || !vs || !pgadv) { set_error("null argument"); return CB_EINVAL; }
  return launch_vtrace(T, B, V, 1, r, d, logpi, logmu, gamma, lambda_, rho_bar, c_bar, rho_pg_bar, vs, pgadv, rho, (cudaStream_t)stream);
}
int cb_gae(int T, int B, const float* V, const float* r, const uint8_t* d, float gamma, float lambda_, float* adv, float* ret, void* stream) {
  if (T < 0 || B < 0) { set_error("bad argument"); return CB_EINVAL; }
  if (T == 0 || B == 0) return CB_OK;
  if (!V || !r || !d || !adv || !ret) { set_error("null argument"); return CB_EINVAL; }
  return launch_gae(T, B, V, 1, r, d, gamma, lambda_, adv, ret, (cudaStream_t)stream);
}
size_t cb_loss_scratch_bytes(int N) { return 256 + (size_t)(((N < 0 ? 0 : N) + 127) / 128) * 40; }
int cb_impala_loss(int N, int A, const float* head, const int32_t* actions, const float* vs, const float* pgadv, const float* rho, float vf_coef,
                   float ent_coef, int loss_reduction, int precision, void* dhead, float* stats, void* scratch, void* stream) {
  if (N < 0 || A < 1 || A > 31 || check_prec(precision)) { set_error("bad argument"); return CB_EINVAL; }
  if (N == 0) return CB_OK;
  if (!head || !actions || !vs || !pgadv || !dhead || !stats || !scratch || misaligned(scratch, 16)) { set_error("null or misaligned argument"); return CB_EINVAL; }
  double* red = (double*)scratch; float* terms = nullptr;
  return launch_impala_loss(precision, N, A, head, actions, vs, pgadv, rho, vf_coef, ent_coef, loss_reduction, dhead, terms, red, stats, (cudaStream_t)stream);
}
int cb_ppo_loss(int m, int A, const float* head, const int32_t* idx, const int32_t* actions, const float* adv, const float* ret, const float* logp_old,
                float clip_eps, float vf_coef, float ent_coef, int norm_adv, int precision, void* dhead, float* stats, void* scratch, void* stream) {
  if (m < 0 || A < 1 || A > 31 || check_prec(precision)) { set_error("bad argument"); return CB_EINVAL; }
  if (m == 0) return CB_OK;
  if (!head || !actions || !adv || !ret || !logp_old || !dhead || !stats || !scratch || misaligned(scratch, 16)) { set_error("null or misaligned argument"); return CB_EINVAL; }
  double* red = (double*)scratch; float* terms = nullptr;
  return launch_ppo_loss(precision, m, A, head, idx, actions, adv, ret, logp_old, clip_eps, vf_coef, ent_coef, norm_adv, dhead, terms, red, nullptr, stats, (cudaStream_t)stream);
}
int cb_permutation(uint64_t seed, uint32_t epoch, int N, int32_t* perm, void* stream) {
  if (N < 0 || !perm) { set_error("bad argument"); return CB_EINVAL; }
  if (N == 0) return CB_OK;
  uint32_t* jb = nullptr;
  CB_CUDA(cudaMallocAsync((void**)&jb, (size_t)N * 4, (cudaStream_t)stream));
  int rc = launch_permutation(seed, epoch, 1, N, perm, jb, (cudaStream_t)stream);
  cudaFreeAsync(jb, (cudaStream_t)stream);
  return rc;
}
int cb_permutation_ws(uint64_t seed, uint32_t epoch, int N, int32_t* perm, uint32_t* scratch, void* stream) {
  if (N < 0 || !perm || (!scratch && N > 0)) { set_error("bad argument"); return CB_EINVAL; }
  if (N == 0) return CB_OK;
  return launch_permutation(seed, epoch, 1, N, perm, scratch, (cudaStream_t)stream);
}
int cb_clip_rmsprop(size_t P, float* params, float* nu, const float* grad, float lr, float decay, float eps, float max_norm, float* grad_norm,
                    void* scratch, void* stream) {
  if (!params || !nu || !grad || !scratch) { set_error("bad argument"); return CB_EINVAL; }
  if (misaligned(params, 16) || misaligned(nu, 16) || misaligned(grad, 16) || misaligned(scratch, 8)) { set_error("buffers must be 16-byte aligned"); return CB_EINVAL; }
  return launch_clip_rmsprop(P, params, nu, grad, lr, decay, eps, max_norm, grad_norm, nullptr, scratch, (cudaStream_t)stream);
}
float cb_linear_lr(float lr0, uint64_t k, uint64_t total) {
  if (total == 0) return lr0;
  return (float)((double)lr0 * (1.0 - (double)std::min(k, total) / (double)total));
}
size_t cb_clip_adam_scratch_bytes(size_t P) { return clip_adam_scratch_bytes(P); }
int cb_clip_adam(size_t P, float* params, float* adam_m, float* adam_v, const float* grad, uint64_t k, float lr, float beta1, float beta2,
                 float eps, float max_norm, float* grad_norm, void* scratch, void* stream) {
  if (!params || !adam_m || !adam_v || !grad || !scratch || k < 1) { set_error("bad argument"); return CB_EINVAL; }
  if (misaligned(params, 16) || misaligned(adam_m, 16) || misaligned(adam_v, 16) || misaligned(grad, 16) || misaligned(scratch, 8)) { set_error("buffers must be 16-byte aligned"); return CB_EINVAL; }
  return launch_clip_adam(P, params, adam_m, adam_v, grad, k, lr, beta1, beta2, eps, max_norm, grad_norm, nullptr, scratch, (cudaStream_t)stream);
}

}  // extern "C"
