"""ctypes loader for the CPU oracle (oracle/cleanba_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, bench.py's cpu_baseline / --impl reference leg and __graft_entry__.smoke() may
import this module.  It never imports the CUDA package and shares no code with it.
All arrays are host numpy arrays; see the .cpp for the citation of every function.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cleanba_oracle.cpp")
_SO = os.path.join(_HERE, "libcleanba_oracle.so")
N_STATS = 8
STAT_NAMES = ("loss", "pg_loss", "v_loss", "entropy", "grad_norm", "approx_kl", "clip_frac", "mean_rho")


def build(force=False):
    """g++ -O2, no fast-math, no fp contraction (fixed_log needs exactly the fma calls it writes)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-ffp-contract=off",
                               "-fno-fast-math", "-o", _SO, _SRC])
    return _SO


class Arch(C.Structure):
    _fields_ = [("kind", C.c_int), ("in_c", C.c_int), ("in_h", C.c_int), ("in_w", C.c_int),
                ("channels", C.c_int * 3), ("fc", C.c_int), ("n_actions", C.c_int)]


class HParams(C.Structure):
    _fields_ = [("algo", C.c_int), ("T", C.c_int), ("B", C.c_int),
                ("gamma", C.c_double), ("lambda_", C.c_double),
                ("rho_bar", C.c_double), ("c_bar", C.c_double), ("rho_pg_bar", C.c_double),
                ("clip_eps", C.c_double), ("epochs", C.c_int), ("minibatches", C.c_int), ("norm_adv", C.c_int),
                ("perm_seed", C.c_uint64),
                ("vf_coef", C.c_double), ("ent_coef", C.c_double),
                ("lr", C.c_double), ("beta1", C.c_double), ("beta2", C.c_double), ("adam_eps", C.c_double),
                ("max_grad_norm", C.c_double), ("loss_reduction", C.c_int),
                ("optimizer", C.c_int), ("rms_decay", C.c_double), ("rms_eps", C.c_double)]


def make_arch(kind, channels, fc, n_actions=18, in_c=4, in_h=84, in_w=84):
    a = Arch(); a.kind = {"nature": 0, "impala": 1}.get(kind, kind)
    a.in_c, a.in_h, a.in_w = in_c, in_h, in_w
    a.channels[:] = list(channels); a.fc = fc; a.n_actions = n_actions
    return a


def make_hparams(algo="impala", T=20, B=128, **kw):
    """Defaults are Table 3 (IMPALA) / Table 2 (PPO) with
    BASELINE.json's Adam for IMPALA (reading A12)."""
    h = HParams(); ppo = algo in ("ppo", 1)
    h.algo = 1 if ppo else 0; h.T = T; h.B = B
    h.gamma = 0.99; h.lambda_ = 0.95 if ppo else 1.0
    h.rho_bar = h.c_bar = h.rho_pg_bar = 1.0
    h.clip_eps = 0.1; h.epochs = 4; h.minibatches = 4 if ppo else 1; h.norm_adv = 1; h.perm_seed = 1
    h.optimizer = 0; h.rms_decay = 0.99; h.rms_eps = 0.01          # Table 3; optimizer 1 = RMSprop (A22)
    h.vf_coef = 0.5; h.ent_coef = 0.01
    h.lr = 2.5e-4 if ppo else 6e-4; h.beta1 = 0.9; h.beta2 = 0.999; h.adam_eps = 1e-5
    h.max_grad_norm = 0.5 if ppo else 40.0; h.loss_reduction = 0
    for k, v in kw.items():
        if not hasattr(h, k):
            raise KeyError(k)
        setattr(h, k, v)
    return h


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_param_count.restype = C.c_size_t
        _lib.orc_fixed_log.restype = C.c_double; _lib.orc_fixed_log.argtypes = [C.c_double]
        _lib.orc_gumbel_from_u32.restype = C.c_float; _lib.orc_gumbel_from_u32.argtypes = [C.c_uint32]
        _lib.orc_clip_adam.restype = C.c_double
        _lib.orc_clip_rmsprop.restype = C.c_double
        _lib.orc_linear_lr.restype = C.c_double
        _lib.orc_impala_objective_f64.restype = C.c_double
        _lib.orc_ppo_objective_f64.restype = C.c_double
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _c(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


def param_count(arch):
    return int(lib().orc_param_count(C.byref(arch)))


def param_tensors(arch):
    """[(offset, count, fan_in)] in canonical order."""
    out, i = [], 0
    off, cnt, fan = C.c_size_t(), C.c_size_t(), C.c_int()
    while lib().orc_param_tensor(C.byref(arch), C.c_int(i), C.byref(off), C.byref(cnt), C.byref(fan)):
        out.append((off.value, cnt.value, fan.value)); i += 1
    return out


def feature_shape(arch):
    c, h, w = C.c_int(), C.c_int(), C.c_int()
    lib().orc_feature_shape(C.byref(arch), C.byref(c), C.byref(h), C.byref(w))
    return c.value, h.value, w.value


def forward(arch, params, obs):
    """params f32 [P], obs u8 [F,C,H,W] -> (logits f64 [F,A], values f64 [F])."""
    params = _c(params, np.float32); obs = _c(obs, np.uint8); F = obs.shape[0]
    lg = np.empty((F, arch.n_actions), np.float64); v = np.empty(F, np.float64)
    lib().orc_forward(C.byref(arch), _p(params), _p(obs), C.c_int(F), _p(lg), _p(v), None, None)
    return lg, v


def forward_f32(arch, params, obs):
    """ABI-rounded outputs: logits f32 [F,A], values f32 [F]."""
    params = _c(params, np.float32); obs = _c(obs, np.uint8); F = obs.shape[0]
    lg = np.empty((F, arch.n_actions), np.float32); v = np.empty(F, np.float32)
    lib().orc_forward(C.byref(arch), _p(params), _p(obs), C.c_int(F), None, None, _p(lg), _p(v))
    return lg, v


def forward_f64(arch, params64, obs):
    params64 = _c(params64, np.float64); obs = _c(obs, np.uint8); F = obs.shape[0]
    lg = np.empty((F, arch.n_actions), np.float64); v = np.empty(F, np.float64)
    lib().orc_forward_f64(C.byref(arch), _p(params64), _p(obs), C.c_int(F), _p(lg), _p(v))
    return lg, v


def backward_f64(arch, params64, obs, dlogits, dV):
    params64 = _c(params64, np.float64); obs = _c(obs, np.uint8); F = obs.shape[0]
    dlogits = _c(dlogits, np.float64); dV = _c(dV, np.float64)
    g = np.zeros(params64.shape[0], np.float64)
    lib().orc_backward_f64(C.byref(arch), _p(params64), _p(obs), C.c_int(F), _p(dlogits), _p(dV), _p(g))
    return g


def log_softmax(logits):
    logits = _c(logits, np.float64); F, A = logits.shape
    lp = np.empty((F, A), np.float64); H = np.empty(F, np.float64)
    lib().orc_log_softmax(_p(logits), C.c_int(F), C.c_int(A), _p(lp), _p(H))
    return lp, H


def maxpool_same(x):
    x = _c(x, np.float64); Cc, H, W = x.shape; Ho, Wo = (H + 1) // 2, (W + 1) // 2
    y = np.empty((Cc, Ho, Wo)); arg = np.empty((Cc, Ho, Wo), np.int32)
    lib().orc_maxpool_same(_p(x), C.c_int(Cc), C.c_int(H), C.c_int(W), _p(y), _p(arg))
    return y, arg


def philox(ctr, key):
    ctr = _c(ctr, np.uint32); key = _c(key, np.uint32); out = np.empty(4, np.uint32)
    lib().orc_philox4x32_10(_p(ctr), _p(key), _p(out))
    return out


def fixed_log(x):
    return float(lib().orc_fixed_log(C.c_double(x)))


def fixed_log_u24(lo, n):
    out = np.empty(n, np.float64)
    lib().orc_fixed_log_u24(C.c_uint32(lo), C.c_uint32(n), _p(out))
    return out


def gumbel_table(lo, n):
    out = np.empty(n, np.float32)
    lib().orc_gumbel_table(C.c_uint32(lo), C.c_uint32(n), _p(out))
    return out


def sample(logits_f32, seed, step, env_offset=0):
    lg = _c(logits_f32, np.float32); B, A = lg.shape
    act = np.empty(B, np.int32)
    lib().orc_sample(_p(lg), C.c_int(B), C.c_int(A), C.c_uint64(seed), C.c_uint64(step), C.c_uint32(env_offset), _p(act))
    return act


def permutation(seed, epoch, N):
    perm = np.empty(N, np.int32)
    lib().orc_permutation(C.c_uint64(seed), C.c_uint32(epoch), C.c_int(N), _p(perm))
    return perm


def vtrace(V, r, d, logpi, logmu, gamma=0.99, lam=1.0, rho_bar=1.0, c_bar=1.0, rho_pg_bar=1.0):
    """V [T+1,B]; r, d, logpi, logmu [T,B] -> vs, pgadv, rho [T,B] (fp64)."""
    V = _c(V, np.float64); r = _c(r, np.float64); d = _c(d, np.uint8)
    logpi = _c(logpi, np.float64); logmu = _c(logmu, np.float64); T, B = r.shape
    vs = np.empty((T, B)); pg = np.empty((T, B)); rho = np.empty((T, B))
    lib().orc_vtrace(C.c_int(T), C.c_int(B), _p(V), _p(r), _p(d), _p(logpi), _p(logmu), C.c_double(gamma), C.c_double(lam),
                     C.c_double(rho_bar), C.c_double(c_bar), C.c_double(rho_pg_bar), _p(vs), _p(pg), _p(rho))
    return vs, pg, rho


def gae(V, r, d, gamma=0.99, lam=0.95):
    V = _c(V, np.float64); r = _c(r, np.float64); d = _c(d, np.uint8); T, B = r.shape
    adv = np.empty((T, B)); ret = np.empty((T, B))
    lib().orc_gae(C.c_int(T), C.c_int(B), _p(V), _p(r), _p(d), C.c_double(gamma), C.c_double(lam), _p(adv), _p(ret))
    return adv, ret


def impala_loss(logits, V, act, vs, pgadv, rho=None, c1=0.5, c2=0.01, reduction=0):
    logits = _c(logits, np.float64); N, A = logits.shape
    V = _c(V, np.float64); act = _c(act, np.int32); vs = _c(vs, np.float64); pgadv = _c(pgadv, np.float64)
    rho = None if rho is None else _c(rho, np.float64)
    st = np.zeros(N_STATS); dl = np.empty((N, A)); dV = np.empty(N)
    lib().orc_impala_loss(C.c_int(N), C.c_int(A), _p(logits), _p(V), _p(act), _p(vs), _p(pgadv), _p(rho),
                          C.c_double(c1), C.c_double(c2), C.c_int(reduction), _p(st), _p(dl), _p(dV))
    return st, dl, dV


def ppo_loss(logits, V, act, adv, ret, logp_old, eps=0.1, c1=0.5, c2=0.01, norm_adv=1):
    logits = _c(logits, np.float64); m, A = logits.shape
    V = _c(V, np.float64); act = _c(act, np.int32); adv = _c(adv, np.float64); ret = _c(ret, np.float64)
    logp_old = _c(logp_old, np.float64)
    st = np.zeros(N_STATS); dl = np.empty((m, A)); dV = np.empty(m)
    lib().orc_ppo_loss(C.c_int(m), C.c_int(A), _p(logits), _p(V), _p(act), _p(adv), _p(ret), _p(logp_old),
                       C.c_double(eps), C.c_double(c1), C.c_double(c2), C.c_int(norm_adv), _p(st), _p(dl), _p(dV))
    return st, dl, dV


def clip_adam(theta, m, v, g, k, lr, b1=0.9, b2=0.999, eps=1e-5, max_norm=40.0):
    """Returns (theta', m', v', pre-clip norm); inputs untouched."""
    theta = _c(theta, np.float32).copy(); m = _c(m, np.float32).copy(); v = _c(v, np.float32).copy()
    g = _c(g, np.float64)
    n = lib().orc_clip_adam(C.c_size_t(theta.size), _p(theta), _p(m), _p(v), _p(g), C.c_uint64(k), C.c_double(lr),
                            C.c_double(b1), C.c_double(b2), C.c_double(eps), C.c_double(max_norm))
    return theta, m, v, float(n)


def clip_rmsprop(theta, nu, g, lr, decay=0.99, eps=0.01, max_norm=40.0):
    """A22.  Returns (theta', nu', pre-clip norm); inputs untouched."""
    theta = _c(theta, np.float32).copy(); nu = _c(nu, np.float32).copy(); g = _c(g, np.float64)
    n = lib().orc_clip_rmsprop(C.c_size_t(theta.size), _p(theta), _p(nu), _p(g), C.c_double(lr), C.c_double(decay), C.c_double(eps), C.c_double(max_norm))
    return theta, nu, float(n)


def linear_lr(lr0, k, total):
    return float(lib().orc_linear_lr(C.c_double(lr0), C.c_uint64(k), C.c_uint64(total)))


def impala_objective_f64(arch, hp, params64, params_tgt64, obs, actions, rewards, dones, behaviour_logits, want_grad=False):
    params64 = _c(params64, np.float64); params_tgt64 = _c(params_tgt64, np.float64)
    obs = _c(obs, np.uint8); actions = _c(actions, np.int32); rewards = _c(rewards, np.float32)
    dones = _c(dones, np.uint8); bl = _c(behaviour_logits, np.float32)
    g = np.zeros(params64.size) if want_grad else None
    L = lib().orc_impala_objective_f64(C.byref(arch), C.byref(hp), _p(params64), _p(params_tgt64), _p(obs), _p(actions),
                                       _p(rewards), _p(dones), _p(bl), _p(g))
    return (float(L), g) if want_grad else float(L)


def ppo_objective_f64(arch, hp, params64, obs, actions, adv, ret, logp_old, want_grad=False):
    params64 = _c(params64, np.float64); obs = _c(obs, np.uint8); actions = _c(actions, np.int32)
    adv = _c(adv, np.float64); ret = _c(ret, np.float64); logp_old = _c(logp_old, np.float64)
    g = np.zeros(params64.size) if want_grad else None
    L = lib().orc_ppo_objective_f64(C.byref(arch), C.byref(hp), _p(params64), _p(obs), C.c_int(obs.shape[0]), _p(actions),
                                    _p(adv), _p(ret), _p(logp_old), _p(g))
    return (float(L), g) if want_grad else float(L)


def learner_step(arch, hp, params, adam_m, adam_v, opt_step, obs, actions, rewards, dones, behaviour_logits, debug=False,
                 behaviour_values=None):
    """One cb_learner_step on the host.  Returns dict(params, m, v, opt_step, stats[, logits, values, t0, t1, grad])."""
    T, B, A = hp.T, hp.B, arch.n_actions
    params = _c(params, np.float32).copy(); m = _c(adam_m, np.float32).copy(); v = _c(adam_v, np.float32).copy()
    obs = _c(obs, np.uint8); actions = _c(actions, np.int32); rewards = _c(rewards, np.float32)
    dones = _c(dones, np.uint8); bl = _c(behaviour_logits, np.float32)
    assert obs.shape[0] == (T + 1) * B or obs.shape[:2] == (T + 1, B)
    n_upd = max(1, hp.minibatches) if hp.algo == 0 else hp.epochs * hp.minibatches
    stats = np.zeros((n_upd, N_STATS), np.float32); step = C.c_uint64(opt_step)
    F, N = (T + 1) * B, T * B
    dbg = dict(logits=np.empty((F, A)), values=np.empty(F), t0=np.empty(N), t1=np.empty(N), grad=np.empty(params.size)) if debug else {}
    bv = None if behaviour_values is None else _c(behaviour_values, np.float32)
    assert bv is None or bv.size == F
    n = lib().orc_learner_step(C.byref(arch), C.byref(hp), _p(params), _p(m), _p(v), C.byref(step), _p(obs), _p(actions),
                               _p(rewards), _p(dones), _p(bl), _p(bv), _p(stats), _p(dbg.get("logits")), _p(dbg.get("values")),
                               _p(dbg.get("t0")), _p(dbg.get("t1")), _p(dbg.get("grad")))
    assert n == n_upd
    out = dict(params=params, m=m, v=v, opt_step=step.value, stats=stats)
    out.update(dbg)
    return out
