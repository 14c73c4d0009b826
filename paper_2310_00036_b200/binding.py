"""Thin ctypes binding over the C-ABI CUDA library (include/cleanba.h).  Argument marshalling
only: every step of the path runs in the library's kernels.  torch is used for device memory and
streams.  There is NO CPU fallback: a missing library or a missing GPU raises.
"""
import ctypes as C
import os

import numpy as np

from .synth import ArchSpec

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libcleanba.so")
N_STATS = 8
STAT_NAMES = ("loss", "pg_loss", "v_loss", "entropy", "grad_norm", "approx_kl", "clip_frac", "mean_rho")
PREC = {"fp32": 0, "bf16": 1}
ALGO = {"impala": 0, "ppo": 1}

EXPORTS = ["cb_net_create", "cb_net_destroy", "cb_param_count", "cb_param_layout", "cb_net_init", "cb_policy_forward",
           "cb_learner_step", "cb_learner_view", "cb_sample_actions", "cb_logprob_entropy", "cb_vtrace", "cb_gae",
           "cb_permutation", "cb_clip_adam_scratch_bytes", "cb_clip_adam", "cb_last_error",
           "cb_launch_count", "cb_profile_begin", "cb_profile_end", "cb_clip_rmsprop", "cb_linear_lr",
           "cb_learner_begin", "cb_learner_grad", "cb_learner_apply", "cb_sum_ranks", "cb_check_errors",
           "cb_debug_inject_timeout", "cb_permutation_ws", "cb_permutation_static",
           "cb_pipeline_create", "cb_pipeline_destroy", "cb_pipeline_run", "cb_pipeline_wait", "cb_pipeline_state", "cb_pipeline_records",
           "cb_pipeline_rollout", "cb_pipeline_policy_version", "cb_env_state_ints", "cb_env_reset", "cb_env_step",
           "cb_loss_scratch_bytes", "cb_impala_loss", "cb_ppo_loss"]


class CArch(C.Structure):
    _fields_ = [("kind", C.c_int), ("in_c", C.c_int), ("in_h", C.c_int), ("in_w", C.c_int),
                ("channels", C.c_int * 3), ("fc", C.c_int), ("n_actions", C.c_int)]


class CHParams(C.Structure):
    _fields_ = [("algo", C.c_int), ("precision", C.c_int), ("T", C.c_int), ("B", C.c_int),
                ("gamma", C.c_float), ("lambda_", C.c_float),
                ("rho_bar", C.c_float), ("c_bar", C.c_float), ("rho_pg_bar", C.c_float),
                ("clip_eps", C.c_float), ("epochs", C.c_int), ("minibatches", C.c_int), ("norm_adv", C.c_int),
                ("perm_seed", C.c_uint64),
                ("vf_coef", C.c_float), ("ent_coef", C.c_float),
                ("lr", C.c_float), ("beta1", C.c_float), ("beta2", C.c_float), ("adam_eps", C.c_float),
                ("max_grad_norm", C.c_float), ("loss_reduction", C.c_int),
                ("optimizer", C.c_int), ("rms_decay", C.c_float), ("rms_eps", C.c_float)]


class CleanbaError(RuntimeError):
    pass


_lib = None


def lib():
    """Loads libcleanba.so (built in-tree by paper_2310_00036_b200/build.py).  Raises if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise CleanbaError(f"{_SO} is missing: run `python -m paper_2310_00036_b200.build` (no CPU fallback exists)")
        L = C.CDLL(_SO)
        L.cb_param_count.restype = C.c_size_t
        L.cb_clip_adam_scratch_bytes.restype = C.c_size_t
        L.cb_clip_adam_scratch_bytes.argtypes = [C.c_size_t]
        L.cb_last_error.restype = C.c_char_p
        L.cb_launch_count.restype = C.c_uint64
        L.cb_linear_lr.restype = C.c_float
        L.cb_linear_lr.argtypes = [C.c_float, C.c_uint64, C.c_uint64]
        L.cb_net_destroy.restype = None
        L.cb_net_destroy.argtypes = [C.c_void_p]
        L.cb_pipeline_destroy.restype = None
        L.cb_pipeline_destroy.argtypes = [C.c_void_p]
        L.cb_env_state_ints.restype = C.c_size_t
        L.cb_loss_scratch_bytes.restype = C.c_size_t
        _lib = L
    return _lib


def _check(rc):
    if rc < 0:
        raise CleanbaError(f"cleanba error {rc}: {lib().cb_last_error().decode()}")
    return rc


def make_hparams(algo="impala", precision="bf16", T=20, B=128, **kw):
    """Defaults: Table 3 (IMPALA) / Table 2 (PPO); Adam for both (A12)."""
    h = CHParams(); ppo = algo in ("ppo", 1)
    h.algo = 1 if ppo else 0; h.precision = PREC.get(precision, precision); h.T = T; h.B = B
    h.gamma = 0.99; h.lambda_ = 0.95 if ppo else 1.0
    h.rho_bar = h.c_bar = h.rho_pg_bar = 1.0
    h.clip_eps = 0.1; h.epochs = 4; h.minibatches = 4 if ppo else 1; h.norm_adv = 1; h.perm_seed = 1
    h.optimizer = 0; h.rms_decay = 0.99; h.rms_eps = 0.01        # optimizer 1 = the paper's RMSprop (Table 3)
    h.vf_coef = 0.5; h.ent_coef = 0.01
    h.lr = 2.5e-4 if ppo else 6e-4; h.beta1 = 0.9; h.beta2 = 0.999; h.adam_eps = 1e-5
    h.max_grad_norm = 0.5 if ppo else 40.0; h.loss_reduction = 0
    for k, v in kw.items():
        if not hasattr(h, k):
            raise KeyError(k)
        setattr(h, k, v)
    return h


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise CleanbaError("no CUDA device: the Cleanba hot path has no CPU fallback")
    return torch


def _ptr(t):
    return C.c_void_p(0 if t is None else t.data_ptr())


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev(t, dtype, name):
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise CleanbaError(f"{name} must be a contiguous CUDA tensor of dtype {dtype}")
    return t


class Net:
    """cb_net handle.  Creating it and cb_net_init need no GPU; everything else does."""

    def __init__(self, arch: ArchSpec, max_frames=0):
        a = _arch_struct(arch)
        self.arch = arch; self._h = C.c_void_p()
        _check(lib().cb_net_create(C.byref(a), C.c_int(max_frames), C.byref(self._h)))
        self.P = int(lib().cb_param_count(self._h)); self.A = arch.n_actions

    def close(self):
        if self._h:
            lib().cb_net_destroy(self._h); self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def param_layout(self):
        """[(name, offset, dims)] in canonical order."""
        out, i = [], 0
        name = C.c_char_p(); off = C.c_size_t(); rank = C.c_int(); dims = (C.c_int * 4)()
        while lib().cb_param_layout(self._h, C.c_int(i), C.byref(name), C.byref(off), C.byref(rank), dims) == 0:
            out.append((name.value.decode(), off.value, tuple(dims[:rank.value]))); i += 1
        return out

    def init_params(self, seed):
        """cb_net_init: host He-normal init -> numpy fp32 [P]."""
        p = np.empty(self.P, np.float32)
        _check(lib().cb_net_init(self._h, C.c_uint64(seed), p.ctypes.data_as(C.c_void_p)))
        return p

    def policy_forward(self, params, obs, seed=0, step=0, env_offset=0, precision="bf16", want_actions=True):
        """cb_policy_forward on the current torch stream.  params: cuda fp32 [P], or None to reuse the weights packed by the
        previous call in this precision mode; obs: cuda uint8 [B,C,H,W].  Returns (logits [B,A], value [B], actions int32 [B])."""
        torch = _torch()
        if params is not None:
            _dev(params, torch.float32, "params")
        _dev(obs, torch.uint8, "obs")
        B = obs.shape[0]
        logits = torch.empty((B, self.A), dtype=torch.float32, device=obs.device)
        value = torch.empty((B,), dtype=torch.float32, device=obs.device)
        actions = torch.empty((B,), dtype=torch.int32, device=obs.device) if want_actions else None
        _check(lib().cb_policy_forward(self._h, _ptr(params), _ptr(obs), C.c_int(B), C.c_uint64(seed), C.c_uint64(step),
                                       C.c_uint32(env_offset), C.c_int(PREC.get(precision, precision)), _ptr(logits), _ptr(value),
                                       _ptr(actions), _stream()))
        return logits, value, actions

    def _learner_args(self, params, adam_m, adam_v, obs, actions, rewards, dones, behaviour_logits, behaviour_values, hp, stats):
        torch = _torch()
        for t, n in ((params, "params"), (adam_m, "adam_m"), (adam_v, "adam_v"), (rewards, "rewards"), (behaviour_logits, "behaviour_logits")):
            _dev(t, torch.float32, n)
        _dev(obs, torch.uint8, "obs"); _dev(dones, torch.uint8, "dones"); _dev(actions, torch.int32, "actions")
        if behaviour_values is not None:
            _dev(behaviour_values, torch.float32, "behaviour_values")
        n_upd = hp.epochs * hp.minibatches if hp.algo == 1 else max(1, hp.minibatches)
        if stats is None:
            stats = torch.zeros((n_upd, N_STATS), dtype=torch.float32, device=obs.device)
        return n_upd, stats

    def learner_step(self, params, adam_m, adam_v, opt_step, obs, actions, rewards, dones, behaviour_logits, hp, stats=None,
                     behaviour_values=None):
        """cb_learner_step on the current torch stream; params/adam_m/adam_v are updated in place.
        behaviour_values: cuda fp32 [T+1,B] actor-time values (PPO, A3b) or None.
        Returns (new opt_step, stats tensor [n_updates, 8])."""
        n_upd, stats = self._learner_args(params, adam_m, adam_v, obs, actions, rewards, dones, behaviour_logits, behaviour_values, hp, stats)
        k = C.c_uint64(opt_step)
        rc = _check(lib().cb_learner_step(self._h, _ptr(params), _ptr(adam_m), _ptr(adam_v), C.byref(k), _ptr(obs), _ptr(actions),
                                          _ptr(rewards), _ptr(dones), _ptr(behaviour_logits), _ptr(behaviour_values), C.byref(hp),
                                          _ptr(stats), _stream()))
        assert rc == n_upd
        return k.value, stats

    def learner_begin(self, params, adam_m, adam_v, opt_step, obs, actions, rewards, dones, behaviour_logits, hp, stats=None,
                      behaviour_values=None):
        """cb_learner_begin.  Returns (n_updates, stats, handle); the handle keeps every buffer (and the host step counter)
        alive until the last learner_apply; handle.opt_step is the running update count."""
        n_upd, stats = self._learner_args(params, adam_m, adam_v, obs, actions, rewards, dones, behaviour_logits, behaviour_values, hp, stats)
        h = _LearnHandle(C.c_uint64(opt_step), (params, adam_m, adam_v, obs, actions, rewards, dones, behaviour_logits, behaviour_values, hp, stats))
        rc = _check(lib().cb_learner_begin(self._h, _ptr(params), _ptr(adam_m), _ptr(adam_v), C.byref(h.k), _ptr(obs), _ptr(actions),
                                           _ptr(rewards), _ptr(dones), _ptr(behaviour_logits), _ptr(behaviour_values), C.byref(hp),
                                           _ptr(stats), _stream()))
        assert rc == n_upd
        self._learn = h
        return n_upd, stats, h

    def learner_grad(self, update):
        """cb_learner_grad: computes update `update`'s gradient; returns it as a torch VIEW of the library-owned [P] buffer."""
        torch = _torch()
        g = C.c_void_p()
        _check(lib().cb_learner_grad(self._h, C.c_int(update), C.byref(g), _stream()))
        return torch.as_tensor(_DevView(g.value, self.P), device="cuda")

    def learner_apply(self, update):
        _check(lib().cb_learner_apply(self._h, C.c_int(update), _stream()))
        return self._learn.opt_step

    def check_errors(self):
        """cb_check_errors: synchronises the current stream; raises if a kernel reported a pipeline time-out."""
        _check(lib().cb_check_errors(self._h, _stream()))

    def debug_inject_timeout(self, precision="bf16"):
        _check(lib().cb_debug_inject_timeout(self._h, C.c_int(PREC.get(precision, precision)), _stream()))

    def learner_view(self, which):
        """Copy of a library-owned result of the last learner step (cb_learner_view) as a torch tensor."""
        torch = _torch()
        p = C.c_void_p(); n = C.c_size_t()
        _check(lib().cb_learner_view(self._h, C.c_int(which), C.byref(p), C.byref(n)))
        torch.cuda.current_stream().synchronize()
        return torch.as_tensor(_DevView(p.value, n.value), device="cuda").clone()


class _LearnHandle:
    def __init__(self, k, keep):
        self.k = k; self._keep = keep

    @property
    def opt_step(self):
        return int(self.k.value)


class _DevView:
    """__cuda_array_interface__ holder for a library-owned fp32 device buffer."""

    def __init__(self, ptr, n):
        self.__cuda_array_interface__ = {"shape": (n,), "typestr": "<f4", "data": (ptr, False), "version": 2}


# ---- Cleanba's actor/learner architecture (cb_pipeline_*) and the synthetic environment ------------------
class CPipelineCfg(C.Structure):
    _fields_ = [("sync", C.c_int), ("actor_values", C.c_int), ("serial", C.c_int), ("env_seed", C.c_uint64), ("sample_seed", C.c_uint64)]


class CPipelineRecord(C.Structure):
    _fields_ = [("iteration", C.c_int), ("data_policy_version", C.c_int), ("learner_version_before", C.c_int), ("learner_version_after", C.c_int)]


def _arch_struct(arch):
    a = CArch(); a.kind = {"nature": 0, "impala": 1}[arch.kind]
    a.in_c, a.in_h, a.in_w = arch.in_c, arch.in_h, arch.in_w
    a.channels[:] = list(arch.channels); a.fc = arch.fc; a.n_actions = arch.n_actions
    return a


def pipeline_policy_version(sync, iteration):
    """cb_pipeline_policy_version (host arithmetic, needs no GPU)."""
    return int(lib().cb_pipeline_policy_version(C.c_int(1 if sync else 0), C.c_int(iteration)))


class Pipeline:
    """cb_pipeline handle: actor stream + learner stream with event-ordered double buffers (Figure 1 right / Table 1)."""

    def __init__(self, arch, hp, params, sync=False, actor_values=False, serial=False, env_seed=1, sample_seed=2):
        torch = _torch(); _dev(params, torch.float32, "params")
        cfg = CPipelineCfg(1 if sync else 0, 1 if actor_values else 0, 1 if serial else 0, env_seed, sample_seed)
        a = _arch_struct(arch)
        self.arch, self.hp, self._h = arch, hp, C.c_void_p()
        _check(lib().cb_pipeline_create(C.byref(a), C.byref(hp), C.byref(cfg), _ptr(params), C.byref(self._h)))
        self.T, self.B, self.A = hp.T, hp.B, arch.n_actions
        self.n_upd = hp.epochs * hp.minibatches if hp.algo == 1 else max(1, hp.minibatches)
        self.P = params.numel()

    def close(self):
        if self._h:
            lib().cb_pipeline_destroy(self._h); self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def run(self, iterations):
        _check(lib().cb_pipeline_run(self._h, C.c_int(iterations)))

    def wait(self):
        """Waits for both streams; returns the device time (ms) of the last run()."""
        ms = C.c_float()
        _check(lib().cb_pipeline_wait(self._h, C.byref(ms)))
        return float(ms.value)

    def state(self):
        """(params, adam_m, adam_v) as torch COPIES, opt_step, iterations; waits first."""
        torch = _torch(); self.wait()
        p, m, v = C.c_void_p(), C.c_void_p(), C.c_void_p(); k = C.c_uint64(); it = C.c_int()
        _check(lib().cb_pipeline_state(self._h, C.byref(p), C.byref(m), C.byref(v), C.byref(k), C.byref(it)))
        cp = lambda q: torch.as_tensor(_DevView(q.value, self.P), device="cuda").clone()
        return cp(p), cp(m), cp(v), int(k.value), int(it.value)

    def records(self, max_n=64):
        buf = (CPipelineRecord * max_n)()
        n = _check(lib().cb_pipeline_records(self._h, buf, C.c_int(max_n)))
        return [(r.iteration, r.data_policy_version, r.learner_version_before, r.learner_version_after) for r in buf[:n]]

    def rollout(self, iteration):
        """Copies of the rollout storage D of `iteration` (one of the last two) and of its learner call's stats; waits first."""
        torch = _torch(); self.wait()
        ptr = [C.c_void_p() for _ in range(7)]
        _check(lib().cb_pipeline_rollout(self._h, C.c_int(iteration), *[C.byref(q) for q in ptr]))
        T, B, A, a = self.T, self.B, self.A, self.arch

        def view(q, n, typestr, shape):
            h = _DevView(q.value, n); h.__cuda_array_interface__["typestr"] = typestr
            return torch.as_tensor(h, device="cuda").clone().reshape(shape)
        return dict(obs=view(ptr[0], (T + 1) * B * a.in_c * a.in_h * a.in_w, "|u1", (T + 1, B, a.in_c, a.in_h, a.in_w)),
                    actions=view(ptr[1], T * B, "<i4", (T, B)), rewards=view(ptr[2], T * B, "<f4", (T, B)), dones=view(ptr[3], T * B, "|u1", (T, B)),
                    behaviour_logits=view(ptr[4], T * B * A, "<f4", (T, B, A)), values=view(ptr[5], (T + 1) * B, "<f4", (T + 1, B)),
                    stats=view(ptr[6], self.n_upd * N_STATS, "<f4", (self.n_upd, N_STATS)))


def env_state_ints():
    return int(lib().cb_env_state_ints())


def env_reset(seed, B, arch):
    torch = _torch()
    state = torch.zeros((B, env_state_ints()), dtype=torch.int32, device="cuda")
    obs = torch.empty((B, arch.in_c, arch.in_h, arch.in_w), dtype=torch.uint8, device="cuda")
    _check(lib().cb_env_reset(C.c_uint64(seed), C.c_int(B), C.c_int(arch.in_c), C.c_int(arch.in_h), C.c_int(arch.in_w), _ptr(state), _ptr(obs), _stream()))
    return state, obs


def env_step(seed, global_step, actions, state, obs):
    """In place on `state`; returns (next obs, rewards, dones)."""
    torch = _torch(); _dev(actions, torch.int32, "actions"); _dev(state, torch.int32, "state"); _dev(obs, torch.uint8, "obs")
    B, Cc, H, W = obs.shape
    out = torch.empty_like(obs); rew = torch.empty((B,), dtype=torch.float32, device="cuda"); done = torch.empty((B,), dtype=torch.uint8, device="cuda")
    _check(lib().cb_env_step(C.c_uint64(seed), C.c_int(B), C.c_int(Cc), C.c_int(H), C.c_int(W), C.c_uint32(global_step), _ptr(actions), _ptr(state),
                             _ptr(obs), _ptr(out), _ptr(rew), _ptr(done), _stream()))
    return out, rew, done


# ---- sub-step entry points --------------------------------------------------------------------------
def sample_actions(logits, seed, step, env_offset=0):
    torch = _torch(); _dev(logits, torch.float32, "logits"); B, A = logits.shape
    act = torch.empty((B,), dtype=torch.int32, device=logits.device)
    _check(lib().cb_sample_actions(_ptr(logits), C.c_int(B), C.c_int(A), C.c_uint64(seed), C.c_uint64(step), C.c_uint32(env_offset), _ptr(act), _stream()))
    return act


def logprob_entropy(logits, actions):
    torch = _torch(); _dev(logits, torch.float32, "logits"); _dev(actions, torch.int32, "actions"); N, A = logits.shape
    lp = torch.empty((N,), dtype=torch.float32, device=logits.device); H = torch.empty_like(lp)
    _check(lib().cb_logprob_entropy(_ptr(logits), C.c_int(A), C.c_int(N), C.c_int(A), _ptr(actions), _ptr(lp), _ptr(H), _stream()))
    return lp, H


def vtrace(V, r, d, logpi, logmu, gamma=0.99, lam=1.0, rho_bar=1.0, c_bar=1.0, rho_pg_bar=1.0):
    torch = _torch(); T, B = r.shape
    for t, n in ((V, "V"), (r, "r"), (logpi, "logpi"), (logmu, "logmu")):
        _dev(t, torch.float32, n)
    _dev(d, torch.uint8, "d")
    vs = torch.empty_like(r); pg = torch.empty_like(r); rho = torch.empty_like(r)
    _check(lib().cb_vtrace(C.c_int(T), C.c_int(B), _ptr(V), _ptr(r), _ptr(d), _ptr(logpi), _ptr(logmu), C.c_float(gamma), C.c_float(lam),
                           C.c_float(rho_bar), C.c_float(c_bar), C.c_float(rho_pg_bar), _ptr(vs), _ptr(pg), _ptr(rho), _stream()))
    return vs, pg, rho


def gae(V, r, d, gamma=0.99, lam=0.95):
    torch = _torch(); T, B = r.shape
    _dev(V, torch.float32, "V"); _dev(r, torch.float32, "r"); _dev(d, torch.uint8, "d")
    adv = torch.empty_like(r); ret = torch.empty_like(r)
    _check(lib().cb_gae(C.c_int(T), C.c_int(B), _ptr(V), _ptr(r), _ptr(d), C.c_float(gamma), C.c_float(lam), _ptr(adv), _ptr(ret), _stream()))
    return adv, ret


def _loss_out(head, precision):
    torch = _torch(); _dev(head, torch.float32, "head")
    bf = PREC.get(precision, precision) == 1
    dhead = torch.empty(head.shape, dtype=torch.bfloat16 if bf else torch.float32, device=head.device)
    stats = torch.zeros((N_STATS,), dtype=torch.float32, device=head.device)
    scratch = torch.empty((int(lib().cb_loss_scratch_bytes(C.c_int(head.shape[0]))) + 7) // 8, dtype=torch.float64, device=head.device)
    return dhead, stats, scratch


def impala_loss(head, actions, vs, pgadv, rho, vf_coef=0.5, ent_coef=0.01, loss_reduction=0, precision="fp32", out=None):
    """cb_impala_loss: head cuda fp32 [N, A+1] -> (dhead [N, A+1] in the mode's storage type, stats [8])."""
    dhead, stats, scratch = out if out is not None else _loss_out(head, precision)
    N, A1 = head.shape
    _check(lib().cb_impala_loss(C.c_int(N), C.c_int(A1 - 1), _ptr(head), _ptr(actions), _ptr(vs), _ptr(pgadv), _ptr(rho), C.c_float(vf_coef), C.c_float(ent_coef),
                                C.c_int(loss_reduction), C.c_int(PREC.get(precision, precision)), _ptr(dhead), _ptr(stats), _ptr(scratch), _stream()))
    return dhead, stats


def ppo_loss(head, idx, actions, adv, ret, logp_old, clip_eps=0.1, vf_coef=0.5, ent_coef=0.01, norm_adv=1, precision="fp32", out=None):
    """cb_ppo_loss: head cuda fp32 [m, A+1] (the minibatch's forward), idx int32 [m] or None -> (dhead, stats [8])."""
    dhead, stats, scratch = out if out is not None else _loss_out(head, precision)
    m, A1 = head.shape
    _check(lib().cb_ppo_loss(C.c_int(m), C.c_int(A1 - 1), _ptr(head), _ptr(idx), _ptr(actions), _ptr(adv), _ptr(ret), _ptr(logp_old), C.c_float(clip_eps),
                             C.c_float(vf_coef), C.c_float(ent_coef), C.c_int(norm_adv), C.c_int(PREC.get(precision, precision)), _ptr(dhead), _ptr(stats),
                             _ptr(scratch), _stream()))
    return dhead, stats


def permutation(seed, epoch, N):
    torch = _torch()
    perm = torch.empty((N,), dtype=torch.int32, device="cuda")
    _check(lib().cb_permutation(C.c_uint64(seed), C.c_uint32(epoch), C.c_int(N), _ptr(perm), _stream()))
    return perm


PERM_STATIC_MAX = 65536      # CB_PERM_STATIC_MAX


def permutation_static(seed, epoch, N, out=None):
    """cb_permutation_static: no allocation inside the call (static device scratch, N <= PERM_STATIC_MAX).  `out`: a caller-owned
    int32 [N] device tensor; without it one is allocated HERE, by torch, before the call."""
    torch = _torch()
    perm = out if out is not None else torch.empty((N,), dtype=torch.int32, device="cuda")
    assert perm.dtype == torch.int32 and perm.numel() >= N and perm.is_contiguous()
    _check(lib().cb_permutation_static(C.c_uint64(seed), C.c_uint32(epoch), C.c_int(N), _ptr(perm), _stream()))
    return perm


def sum_ranks(slices, scale=1.0, out=None):
    """cb_sum_ranks: slices cuda fp32 [G, n] -> scale * (sum over G in rank order), cuda fp32 [n]."""
    torch = _torch(); _dev(slices, torch.float32, "slices"); G, n = slices.shape
    if out is None:
        out = torch.empty((n,), dtype=torch.float32, device=slices.device)
    _check(lib().cb_sum_ranks(_ptr(slices), C.c_int(G), C.c_size_t(n), C.c_float(scale), _ptr(out), _stream()))
    return out


def clip_adam(params, adam_m, adam_v, grad, k, lr, beta1=0.9, beta2=0.999, eps=1e-5, max_norm=40.0, scratch=None):
    """In place on params/adam_m/adam_v; returns the pre-clip gradient norm as a cuda fp32 [1] tensor."""
    torch = _torch(); P = params.numel()
    for t, n in ((params, "params"), (adam_m, "adam_m"), (adam_v, "adam_v"), (grad, "grad")):
        _dev(t, torch.float32, n)
    if scratch is None:
        scratch = torch.empty((int(lib().cb_clip_adam_scratch_bytes(C.c_size_t(P))) + 7) // 8, dtype=torch.float64, device=params.device)
    gn = torch.empty((1,), dtype=torch.float32, device=params.device)
    _check(lib().cb_clip_adam(C.c_size_t(P), _ptr(params), _ptr(adam_m), _ptr(adam_v), _ptr(grad), C.c_uint64(k), C.c_float(lr), C.c_float(beta1),
                              C.c_float(beta2), C.c_float(eps), C.c_float(max_norm), _ptr(gn), _ptr(scratch), _stream()))
    return gn


def clip_rmsprop(params, nu, grad, lr, decay=0.99, eps=0.01, max_norm=40.0, scratch=None):
    """In place on params / nu; returns the pre-clip gradient norm as a cuda fp32 [1] tensor (A22)."""
    torch = _torch(); P = params.numel()
    for t, n in ((params, "params"), (nu, "nu"), (grad, "grad")):
        _dev(t, torch.float32, n)
    if scratch is None:
        scratch = torch.empty((int(lib().cb_clip_adam_scratch_bytes(C.c_size_t(P))) + 7) // 8, dtype=torch.float64, device=params.device)
    gn = torch.empty((1,), dtype=torch.float32, device=params.device)
    _check(lib().cb_clip_rmsprop(C.c_size_t(P), _ptr(params), _ptr(nu), _ptr(grad), C.c_float(lr), C.c_float(decay), C.c_float(eps), C.c_float(max_norm),
                                 _ptr(gn), _ptr(scratch), _stream()))
    return gn


def linear_lr(lr0, k, total):
    return float(lib().cb_linear_lr(C.c_float(lr0), C.c_uint64(k), C.c_uint64(total)))


# ---- instrumentation ----------------------------------------------------------------------------------
class CProfEntry(C.Structure):
    _fields_ = [("cls", C.c_int), ("name", C.c_char * 28), ("launches", C.c_uint64), ("ms", C.c_double), ("flops", C.c_double), ("bytes", C.c_double)]


def launch_count():
    return int(lib().cb_launch_count())


def profile_begin(only_class=-1):
    _check(lib().cb_profile_begin(C.c_int(only_class)))


def profile_end():
    """[{cls, name, launches, ms, flops, bytes}] for every kernel class launched since profile_begin (synchronises)."""
    buf = (CProfEntry * 32)()
    n = _check(lib().cb_profile_end(buf, C.c_int(32)))
    return [dict(cls=e.cls, name=e.name.decode(), launches=int(e.launches), ms=e.ms, flops=e.flops, bytes=e.bytes) for e in buf[:n]]
