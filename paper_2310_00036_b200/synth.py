"""Seeded synthetic inputs shared by the CPU oracle's tests and the CUDA path's tests / bench.

This module holds NONE of the method's arithmetic: no network, no V-trace/GAE, no loss, no
optimizer, no Gumbel/Philox sampling.  It only draws inputs (numpy Philox bit generator) with the
shapes and value ranges of the paper's Atari workload (84x84 grey, 4 stacked uint8 frames,
18 actions: PAPER.md:166; unroll 20 / 128, 128 envs: PAPER.md:378-379, 397-398) following the
recipes in DESIGN.md section 4 / SURVEY.md section 8(d).  It imports neither oracle/ nor the
CUDA binding.
"""
from dataclasses import dataclass, field

import numpy as np


@dataclass(frozen=True)
class ArchSpec:
    kind: str = "impala"            # "nature" | "impala"
    channels: tuple = (16, 32, 32)
    fc: int = 256
    n_actions: int = 18
    in_c: int = 4
    in_h: int = 84
    in_w: int = 84


NATURE = ArchSpec("nature", (32, 64, 64), 512)
IMPALA = ArchSpec("impala", (16, 32, 32), 256)
IMPALA_WIDE = ArchSpec("impala", (32, 64, 64), 512)

# BASELINE.json configs[0..4]; seeds = 1000 + index
CONFIGS = {
    0: dict(arch=NATURE, algo="impala", T=5, B=4, precision="fp32", lr=6e-4, max_grad_norm=40.0, obs="uniform"),
    1: dict(arch=IMPALA, algo="actor", T=0, B=128, precision="bf16", obs="blobs"),
    2: dict(arch=IMPALA, algo="impala", T=20, B=128, precision="bf16", lr=6e-4, max_grad_norm=40.0, obs="blobs"),
    3: dict(arch=IMPALA, algo="ppo", T=128, B=64, precision="bf16", lr=2.5e-4, max_grad_norm=0.5, obs="blobs"),
    4: dict(arch=IMPALA_WIDE, algo="impala", T=20, B=1024, precision="bf16", lr=6e-4, max_grad_norm=40.0, obs="blobs"),
}


def rng(seed):
    return np.random.Generator(np.random.Philox(seed))


# ---- shape bookkeeping (layout only; cross-checked against oracle and library in tests) ---------
def _conv_out(h, k, s, p):
    return (h + 2 * p - k) // s + 1


def param_tensors(arch):
    """[(name, shape, fan_in)] in the canonical flat order: stage/layer order, weight then bias;
    conv weights [Cout,Cin,kh,kw]; FC [out,in] with `in` flattened (C,H,W)."""
    out = []; c, h, w = arch.in_c, arch.in_h, arch.in_w

    def conv(name, cout, k, s, p):
        nonlocal c, h, w
        out.append((name + ".w", (cout, c, k, k), c * k * k)); out.append((name + ".b", (cout,), c * k * k))
        h, w, c = _conv_out(h, k, s, p), _conv_out(w, k, s, p), cout

    if arch.kind == "nature":
        conv("conv1", arch.channels[0], 8, 4, 0); conv("conv2", arch.channels[1], 4, 2, 0); conv("conv3", arch.channels[2], 3, 1, 0)
    else:
        for s in range(3):
            conv(f"stage{s}.conv", arch.channels[s], 3, 1, 1)
            h, w = (h + 1) // 2, (w + 1) // 2
            for b in range(2):
                conv(f"stage{s}.block{b}.conv1", arch.channels[s], 3, 1, 1)
                conv(f"stage{s}.block{b}.conv2", arch.channels[s], 3, 1, 1)
    k = c * h * w
    out += [("fc.w", (arch.fc, k), k), ("fc.b", (arch.fc,), k),
            ("pi.w", (arch.n_actions, arch.fc), arch.fc), ("pi.b", (arch.n_actions,), arch.fc),
            ("v.w", (1, arch.fc), arch.fc), ("v.b", (1,), arch.fc)]
    return out


def param_count(arch):
    return int(sum(int(np.prod(s)) for _, s, _ in param_tensors(arch)))


def gen_params(arch, seed, bias_scale=0.0, head_scale=1.0):
    """He-normal weights N(0, 2/fan_in), biases 0 (reading A14) -- or small random biases when
    bias_scale > 0 so that bias-gradient paths are exercised by parity tests.  head_scale < 1 shrinks
    pi.w and v.w so that logits and values are O(1), the regime of an Atari agent trained on rewards
    in {-1,0,+1} (raw He-init heads on unnormalised frames give |V| ~ 10); DESIGN.md section 4."""
    g = rng(seed); parts = []
    for name, shape, fan in param_tensors(arch):
        n = int(np.prod(shape))
        if name.endswith(".w"):
            sc = head_scale if name in ("pi.w", "v.w") else 1.0
            parts.append(g.standard_normal(n) * np.sqrt(2.0 / fan) * sc)
        else:
            parts.append(g.standard_normal(n) * bias_scale)
    return np.concatenate(parts).astype(np.float32)


# ---- observations --------------------------------------------------------------------------------
def gen_obs_uniform(n_frames, seed, arch=NATURE):
    """config 0: i.i.d. uniform{0..255}."""
    return rng(seed).integers(0, 256, size=(n_frames, arch.in_c, arch.in_h, arch.in_w), dtype=np.uint8)


def gen_obs_blobs(T1, B, seed, arch=IMPALA, dones=None):
    """configs 1-4: per env, 8 Gaussian blobs (centre U[0,H)^2, sigma U[3,12] px, amplitude U[40,200])
    drifting with velocity U[-2,2]^2 px/frame; the 4-stack at step t shows frames t..t+3 of that motion
    (a stack shifts by one frame per step); blobs are redrawn after a done; plus integer noise U{0..15};
    clipped to [0,255].  Returns uint8 [T1,B,C,H,W]."""
    g = rng(seed); C, H, W = arch.in_c, arch.in_h, arch.in_w
    yy, xx = np.meshgrid(np.arange(H, dtype=np.float32), np.arange(W, dtype=np.float32), indexing="ij")
    obs = np.empty((T1, B, C, H, W), np.uint8)
    nb = 8

    def draw(n):
        return (g.uniform(0, H, (n, nb, 2)).astype(np.float32), g.uniform(3, 12, (n, nb)).astype(np.float32),
                g.uniform(40, 200, (n, nb)).astype(np.float32), g.uniform(-2, 2, (n, nb, 2)).astype(np.float32))

    cen, sig, amp, vel = draw(B)
    for t in range(T1):
        if dones is not None and t > 0:
            for b in np.nonzero(dones[t - 1])[0]:
                c1, s1, a1, v1 = draw(1); cen[b], sig[b], amp[b], vel[b] = c1[0], s1[0], a1[0], v1[0]
        for c in range(C):
            pos = cen + (t + c) * vel                                           # [B,nb,2]
            d2 = (yy[None, None] - pos[..., 0, None, None]) ** 2 + (xx[None, None] - pos[..., 1, None, None]) ** 2
            img = (amp[..., None, None] * np.exp(-d2 / (2 * sig[..., None, None] ** 2))).sum(1)
            img += g.integers(0, 16, size=(B, H, W))
            obs[t, :, c] = np.clip(img, 0, 255).astype(np.uint8)
    return obs


# ---- trajectories ----------------------------------------------------------------------------------
def gen_rewards_dones(T, B, seed):
    """rewards in {-1,0,+1} w.p. (0.05,0.9,0.05); dones ~ Bernoulli(0.02) (BASELINE.json configs[0])."""
    g = rng(seed)
    rewards = g.choice(np.array([-1.0, 0.0, 1.0], np.float32), size=(T, B), p=[0.05, 0.9, 0.05]).astype(np.float32)
    dones = (g.random((T, B)) < 0.02).astype(np.uint8)
    return rewards, dones


def categorical_from_uniform(logits, u):
    """Inverse-CDF draw from softmax(logits) with given uniforms (generic sampling used to fabricate
    behaviour actions; NOT the method's Gumbel-max sampler)."""
    lg = np.asarray(logits, np.float64); p = np.exp(lg - lg.max(-1, keepdims=True)); p /= p.sum(-1, keepdims=True)
    cdf = np.cumsum(p, -1); a = (u[..., None] > cdf).sum(-1)
    return np.minimum(a, lg.shape[-1] - 1).astype(np.int32)


def gen_behaviour(T, B, A, seed, policy_logits=None, sigma=0.3):
    """behaviour_logits [T,B,A] and actions [T,B].
    config 0: behaviour_logits ~ N(0,1).  configs 2-4 (reading A18): behaviour_logits =
    policy_logits (the caller's forward over obs[:T], whichever implementation it is testing) +
    N(0, sigma) noise; actions are drawn from the BEHAVIOUR softmax."""
    g = rng(seed)
    noise = g.standard_normal((T, B, A)).astype(np.float32)
    u = g.random((T, B))
    bl = noise if policy_logits is None else (np.asarray(policy_logits, np.float32).reshape(T, B, A) + np.float32(sigma) * noise)
    bl = bl.astype(np.float32)
    return bl, categorical_from_uniform(bl, u)


def gen_learner_batch(cfg_index, arch=None, T=None, B=None, forward_fn=None, seed=None):
    """Full input set of cb_learner_step for a BASELINE config (optionally at reduced T/B).
    forward_fn(obs_u8[F,C,H,W]) -> logits [F,A] supplies the current-policy logits for configs 2-4."""
    cfg = CONFIGS[cfg_index]; arch = arch or cfg["arch"]; T = T or cfg["T"]; B = B or cfg["B"]
    seed = 1000 + cfg_index if seed is None else seed
    rewards, dones = gen_rewards_dones(T, B, seed + 1)
    if cfg["obs"] == "uniform":
        obs = gen_obs_uniform((T + 1) * B, seed, arch).reshape(T + 1, B, arch.in_c, arch.in_h, arch.in_w)
        pol = None
    else:
        obs = gen_obs_blobs(T + 1, B, seed, arch, dones)
        pol = None if forward_fn is None else forward_fn(obs[:T].reshape(T * B, arch.in_c, arch.in_h, arch.in_w))
    bl, actions = gen_behaviour(T, B, arch.n_actions, seed + 2, pol)
    return dict(obs=obs, actions=actions, rewards=rewards, dones=dones, behaviour_logits=bl)


# ---- a seeded synthetic ENVIRONMENT (stand-in for EnvPool Atari) -------------------------------------------
# Used by the actor/learner pipeline: `E.step(a_t) -> s_next, r_t, d_next` (Alg. 1 l.9) has to exist on the device so
# that a rollout never leaves it.  This numpy class is the DEFINITION; csrc/env.cu restates it and is tested bit for bit against it.
# Integer arithmetic only (uint32 wrap-around hashes, integer pyramids instead of Gaussians), so "bit for bit" is well defined.
# The world: NB pyramid-shaped blobs on an H x W grey frame.  Blob 0 is the agent's (moved by the action: a % 3 - 1 and (a / 3) % 3 - 1 are
# its x / y direction, actions 0-8 move 2 px, the others 1 px); blobs 1.. drift and bounce.  Touching blob 1 (L1 distance <= 8) pays +1 and
# re-spawns it; touching blob 2 (L1 distance <= 5) pays -1 and ends the episode; an episode also ends with probability 1/64 per step.
# Observations are the last C rendered frames (all C equal after a reset), plus hashed noise in {0..15}: the format of PAPER.md:166.
ENV_NB = 4
ENV_NS = 6 * ENV_NB + 1          # per blob: cx, cy, vx, vy, amp, R; then the episode counter


def mix32(x):
    """32-bit integer mixer (multiply-xorshift); x: uint32 array."""
    x = np.asarray(x, dtype=np.uint64) & 0xFFFFFFFF
    x ^= x >> 16; x = (x * 0x7FEB352D) & 0xFFFFFFFF
    x ^= x >> 15; x = (x * 0x846CA68B) & 0xFFFFFFFF
    x ^= x >> 16
    return x


def env_hash(seed, a, b, c):
    """h(seed, a, b, c) = mix(s ^ mix(a ^ mix(b ^ mix(c)))), s = mix(seed_lo) ^ seed_hi; all uint32, broadcast."""
    s = int(mix32(np.uint64(seed & 0xFFFFFFFF))) ^ ((seed >> 32) & 0xFFFFFFFF)
    a = np.asarray(a, np.uint64) & 0xFFFFFFFF; b = np.asarray(b, np.uint64) & 0xFFFFFFFF; c = np.asarray(c, np.uint64) & 0xFFFFFFFF
    return mix32(np.uint64(s) ^ mix32(a ^ mix32(b ^ mix32(c))))


class BlobEnv:
    """B independent environments.  reset() -> obs uint8 [B,C,H,W]; step(actions int [B], g) -> (obs, reward f32 [B], done u8 [B]) where g
    is the global step counter of the caller (it keys every random draw, so a trajectory is a pure function of (seed, actions))."""

    def __init__(self, B, seed, arch=IMPALA):
        self.B, self.seed, self.C, self.H, self.W = B, seed, arch.in_c, arch.in_h, arch.in_w
        self.state = np.zeros((B, ENV_NS), np.int64)
        self.obs = np.zeros((B, self.C, self.H, self.W), np.uint8)

    def _spawn(self, envs, key):
        """(Re)draw every blob of the listed envs from h(seed, env, key, 8k + field)."""
        e = np.asarray(envs, np.int64)
        for k in range(ENV_NB):
            hh = [env_hash(self.seed, e, key, 8 * k + f).astype(np.int64) for f in range(6)]
            s = self.state
            s[e, 6 * k + 0] = hh[0] % self.W; s[e, 6 * k + 1] = hh[1] % self.H
            s[e, 6 * k + 2] = hh[2] % 5 - 2; s[e, 6 * k + 3] = hh[3] % 5 - 2
            s[e, 6 * k + 4] = 40 + hh[4] % 161; s[e, 6 * k + 5] = 6 + hh[5] % 15

    def _render(self, g):
        B, H, W = self.B, self.H, self.W
        y = np.arange(H, dtype=np.int64)[None, :, None]; x = np.arange(W, dtype=np.int64)[None, None, :]
        img = np.zeros((B, H, W), np.int64)
        for k in range(ENV_NB):
            cx, cy, amp, R = (self.state[:, 6 * k + f][:, None, None] for f in (0, 1, 4, 5))
            img += amp * np.maximum(0, R - np.abs(x - cx)) * np.maximum(0, R - np.abs(y - cy)) // (R * R)
        e = np.arange(B, dtype=np.int64)[:, None, None]
        img += (env_hash(self.seed, e, g, 1000 + y * W + x) & 15).astype(np.int64)
        return np.minimum(img, 255).astype(np.uint8)

    def reset(self):
        self.state[:] = 0
        self._spawn(np.arange(self.B), 0xFFFFFFFF)
        self.obs[:] = self._render(0xFFFFFFFF)[:, None]
        return self.obs.copy()

    def step(self, actions, g):
        s = self.state; B, H, W = self.B, self.H, self.W
        a = np.asarray(actions, np.int64); e = np.arange(B, dtype=np.int64)
        speed = np.where(a < 9, 2, 1)
        s[:, 0] = np.clip(s[:, 0] + (a % 3 - 1) * speed, 0, W - 1); s[:, 1] = np.clip(s[:, 1] + ((a // 3) % 3 - 1) * speed, 0, H - 1)
        for k in range(1, ENV_NB):
            for ax, lim in ((0, W), (1, H)):
                p = s[:, 6 * k + ax] + s[:, 6 * k + 2 + ax]
                out = (p < 0) | (p >= lim)
                s[:, 6 * k + 2 + ax] = np.where(out, -s[:, 6 * k + 2 + ax], s[:, 6 * k + 2 + ax])
                s[:, 6 * k + ax] = np.clip(p, 0, lim - 1)
        d1 = np.abs(s[:, 0] - s[:, 6]) + np.abs(s[:, 1] - s[:, 7]); d2 = np.abs(s[:, 0] - s[:, 12]) + np.abs(s[:, 1] - s[:, 13])
        catch = d1 <= 8; hit = d2 <= 5
        s[:, 6] = np.where(catch, env_hash(self.seed, e, g, 100).astype(np.int64) % W, s[:, 6])
        s[:, 7] = np.where(catch, env_hash(self.seed, e, g, 101).astype(np.int64) % H, s[:, 7])
        reward = np.where(hit, -1.0, np.where(catch, 1.0, 0.0)).astype(np.float32)
        done = hit | (env_hash(self.seed, e, g, 102) % 64 == 0)
        if done.any():
            de = np.nonzero(done)[0]
            s[de, ENV_NS - 1] += 1
            self._spawn(de, (np.uint64(g) * np.uint64(2654435761) + s[de, ENV_NS - 1].astype(np.uint64)) & np.uint64(0xFFFFFFFF))
        frame = self._render(g)
        self.obs[:, :-1] = self.obs[:, 1:]; self.obs[:, -1] = frame
        self.obs[done] = frame[done][:, None]
        return self.obs.copy(), reward, done.astype(np.uint8)
