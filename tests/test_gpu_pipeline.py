"""Cleanba's actor/learner architecture on one GPU (Figure 1 right PAPER.md:35-88, Table 1, section 4.2
PAPER.md:140-152, Synchronous variant PAPER.md:174).  The device-side synthetic environment against its numpy definition (bit for bit),
the policy-version schedule against Table 1 (from device-written records), the two-stream execution against a fully serialised one
(bitwise), and every stage of a short run against the oracle."""
import numpy as np
import pytest

from oracle import oracle
from paper_2310_00036_b200 import binding, build, synth
from helpers import close, dev, host, orc_arch, rel_l2

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

SMALL_IMPALA = synth.ArchSpec("impala", (16, 32, 32), 256, 18, 4, 84, 84)
TINY_IMPALA = synth.ArchSpec("impala", (5, 8, 12), 40, 6, 3, 37, 30)


@pytest.fixture(scope="module", autouse=True)
def _built():
    build.build()


@pytest.mark.parametrize("arch,B", [(SMALL_IMPALA, 5), (TINY_IMPALA, 33)])
def test_env_matches_its_numpy_definition_bit_for_bit(arch, B):
    seed = 2 ** 40 + 77
    ref = synth.BlobEnv(B, seed, arch); o_ref = ref.reset()
    state, obs = binding.env_reset(seed, B, arch)
    assert np.array_equal(host(obs), o_ref) and np.array_equal(host(state), ref.state)
    g = synth.rng(3); n_done = 0; n_rew = 0
    for step in range(150):
        a = g.integers(0, arch.n_actions, B).astype(np.int32)
        if step % 3 == 0:
            a[:] = np.where(ref.state[:, 0] < ref.state[:, 6], 5, 3)          # chase blob 1 along x (a % 3 - 1 = +1 / -1, slow)
        o_ref, r_ref, d_ref = ref.step(a, 1000 + step)
        obs, rew, done = binding.env_step(seed, 1000 + step, dev(a), state, obs)
        assert np.array_equal(host(obs), o_ref), step
        assert np.array_equal(host(rew), r_ref) and np.array_equal(host(done), d_ref) and np.array_equal(host(state), ref.state), step
        n_done += int(d_ref.sum()); n_rew += int((r_ref != 0).sum())
    assert n_done > 0 and n_rew > 0                                            # resets and rewards were exercised


def _pipe(arch, algo, prec, T, B, sync, serial=False, actor_values=False, seed=9, **kw):
    hp = binding.make_hparams(algo, prec, T, B, **kw)
    params = synth.gen_params(arch, seed, bias_scale=0.05, head_scale=0.1)
    return binding.Pipeline(arch, hp, dev(params), sync=sync, actor_values=actor_values, serial=serial, env_seed=seed + 1, sample_seed=seed + 2), hp, params


@pytest.mark.parametrize("sync", [False, True])
def test_policy_version_schedule_is_table_1(sync):
    """Table 1: Synchronous: pi_i --D(pi_i)--> pi_{i+1}.  Cleanba: iteration 1 pi_1 --D(pi_1)--> pi_2, iteration 2
    pi_2 --D(pi_1)--> pi_3, and from iteration 3 on pi_i --D(pi_{i-1})--> pi_{i+1} ("the second latest policy").  The records are written by
    the device: the version word travels with the parameter slot the actor read and with the data slot the learner consumed."""
    pipe, hp, _ = _pipe(SMALL_IMPALA, "impala", "bf16", 3, 4, sync)
    pipe.run(3); pipe.run(4)
    rec = pipe.records()
    exp = [(i, i if sync else max(1, i - 1), i, i + 1) for i in range(1, 8)]
    assert rec == exp
    assert [binding.pipeline_policy_version(sync, i) for i in range(1, 8)] == [e[1] for e in exp]
    p, m, v, k, it = pipe.state()
    assert k == 7 and it == 7 and torch.isfinite(p).all()


@pytest.mark.parametrize("algo,prec,sync,av", [("impala", "bf16", False, False), ("impala", "bf16", True, False), ("ppo", "bf16", False, True),
                                              ("impala", "fp32", False, False)])
def test_two_stream_execution_equals_serialised_execution_bitwise(algo, prec, sync, av):
    """The event-ordered double buffers must make the concurrent execution compute exactly what a device-synchronised execution of the same
    schedule computes: parameters, optimizer state and the last rollouts, byte for byte; twice (A16)."""
    kw = dict(epochs=1, minibatches=2) if algo == "ppo" else {}
    outs = []
    for serial in (True, False, False):
        pipe, hp, _ = _pipe(SMALL_IMPALA, algo, prec, 4, 6, sync, serial=serial, actor_values=av, **kw)
        pipe.run(5)
        p, m, v, k, it = pipe.state()
        d = pipe.rollout(5); d4 = pipe.rollout(4)
        outs.append(b"".join(host(t).tobytes() for t in (p, m, v, d["obs"], d["actions"], d["rewards"], d["behaviour_logits"], d["stats"], d4["obs"], d4["stats"])))
        assert np.isfinite(host(d["stats"])).all()
    assert outs[0] == outs[1] == outs[2]


def test_cleanba_and_synchronous_runs_differ_only_from_iteration_3():
    """Iterations 1 and 2 see the same data in both architectures' first rollout; what differs is WHICH policy collects rollout 2 onward."""
    a, _, _ = _pipe(SMALL_IMPALA, "impala", "bf16", 3, 4, False); b, _, _ = _pipe(SMALL_IMPALA, "impala", "bf16", 3, 4, True)
    a.run(1); b.run(1)
    assert host(a.state()[0]).tobytes() == host(b.state()[0]).tobytes()
    assert host(a.rollout(1)["actions"]).tobytes() == host(b.rollout(1)["actions"]).tobytes()
    a.run(1); b.run(1)
    assert host(a.state()[0]).tobytes() != host(b.state()[0]).tobytes()            # rollout 2: pi_1 (Cleanba) vs pi_2 (Synchronous)


@pytest.mark.parametrize("algo,av", [("impala", False), ("ppo", True)])
def test_pipeline_stages_against_the_oracle(algo, av):
    """A short Cleanba-architecture run in fp32 mode, stage by stage: (1) sampled actions = oracle sampling of the logits the actor
    stored (bit exact, A9); (2) stored logits / values = oracle forward with the policy version Table 1 names; (3) environment
    transitions = the numpy definition driven by the stored actions (bit exact); (4) the learner's update of iteration i from that
    storage = oracle.learner_step with pi_i."""
    arch, T, B, iters = TINY_IMPALA, 4, 5, 4
    kw = dict(epochs=1, minibatches=2) if algo == "ppo" else {}
    pipe, hp, params = _pipe(arch, algo, "fp32", T, B, False, actor_values=av, seed=21, **kw)
    ho = oracle.make_hparams(algo, T, B, **kw)
    for f in ("gamma", "lambda_", "rho_bar", "c_bar", "rho_pg_bar", "clip_eps", "vf_coef", "ent_coef", "lr", "beta1", "beta2", "adam_eps", "max_grad_norm"):
        setattr(ho, f, float(getattr(hp, f)))
    oa = orc_arch(arch); P = params.size
    env = synth.BlobEnv(B, 22, arch); o_prev = env.reset()
    versions = {1: (params.copy(), np.zeros(P, np.float32), np.zeros(P, np.float32), 0)}      # version -> (params, m, v, opt_step) per the GPU
    g = 0
    for i in range(1, iters + 1):
        pipe.run(1)
        d = {k: host(t) for k, t in pipe.rollout(i).items()}
        pv = binding.pipeline_policy_version(False, i)
        assert np.array_equal(d["obs"][0], o_prev)
        for t in range(T):
            assert np.array_equal(d["actions"][t], oracle.sample(d["behaviour_logits"][t], 23, g, 0)), (i, t)       # (1)
            rl, rv = oracle.forward(oa, versions[pv][0], d["obs"][t])                                               # (2)
            close(d["behaviour_logits"][t], rl, 1e-5, what="actor logits"); close(d["values"][t], rv, 1e-5, what="actor values")
            o_next, r, dn = env.step(d["actions"][t], g)                                                            # (3)
            assert np.array_equal(d["obs"][t + 1], o_next) and np.array_equal(d["rewards"][t], r) and np.array_equal(d["dones"][t], dn), (i, t)
            g += 1
        o_prev = d["obs"][T]
        if av:
            _, rv = oracle.forward(oa, versions[pv][0], d["obs"][T]); close(d["values"][T], rv, 1e-5, what="v_next")
        p0, m0, v0, k0 = versions[i]                                                                                # (4): learner holds pi_i
        ref = oracle.learner_step(oa, ho, p0, m0, v0, k0, d["obs"], d["actions"], d["rewards"], d["dones"], d["behaviour_logits"],
                                  behaviour_values=d["values"] if av else None)
        p, m, v, k, _ = pipe.state()
        assert k == ref["opt_step"]
        assert rel_l2(host(p), ref["params"]) < 1e-4 and rel_l2(host(v), ref["v"]) < 1e-3
        for u in range(ref["stats"].shape[0]):
            gs, rs = d["stats"][u].astype(np.float64), ref["stats"][u].astype(np.float64)
            srt = 1e-5 if u == 0 else 1e-4
            scale = abs(rs[1]) + abs(rs[2]) + 0.01 * abs(rs[3]) + 1e-2
            for j in (0, 1, 2, 3):
                assert abs(gs[j] - rs[j]) <= srt * (abs(rs[j]) + scale), (i, u, oracle.STAT_NAMES[j], gs[j], rs[j])
        versions[i + 1] = (host(p), host(m), host(v), k)                     # carry the GPU's state forward: each iteration is checked on its own
    assert pipe.records() == [(i, max(1, i - 1), i, i + 1) for i in range(1, iters + 1)]
