"""Parity of the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.
Bit-exact for integer work (actions, permutations); floating point within the tolerances of
BASELINE.json's north_star: 1e-5 relative in CB_PREC_FP32_REF, 2e-2 relative (1e-3 absolute on
targets) in CB_PREC_BF16_TC; parameters 1e-4 / 5e-3 relative L2 per tensor (reading A15)."""
import numpy as np
import pytest

from oracle import oracle
from paper_2310_00036_b200 import binding, build, synth
from helpers import close, dev, host, rel_l2

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module", autouse=True)
def _built():
    build.build()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"


# ---------------------------------------------------------------------------------------------------
# integer / byte work: bit-exact
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("B,A", [(1, 18), (128, 18), (1000, 18), (37, 6), (64, 4), (5, 1), (33, 31)])
def test_sampling_bit_exact(B, A):
    g = synth.rng(B * 100 + A)
    logits = (g.standard_normal((B, A)) * 2).astype(np.float32)
    for seed, step, off in [(0, 0, 0), (12345678901234567, 3, 7), (2 ** 64 - 1, 2 ** 40 + 5, 2 ** 31)]:
        got = host(binding.sample_actions(dev(logits), seed, step, off))
        ref = oracle.sample(logits, seed, step, off)
        assert np.array_equal(got, ref)


def test_sampling_ties_and_dominant_logit():
    logits = np.zeros((64, 18), np.float32); logits[:, 5] = 1e4
    assert (host(binding.sample_actions(dev(logits), 1, 1)) == 5).all()
    logits = np.full((4096, 18), -3.25, np.float32)   # shift invariance: same actions as all-zero logits
    a0 = host(binding.sample_actions(dev(np.zeros_like(logits)), 9, 2))
    a1 = host(binding.sample_actions(dev(logits), 9, 2))
    assert np.array_equal(a0, a1) and np.array_equal(a0, oracle.sample(logits, 9, 2))
    assert len(np.unique(a0)) == 18


@pytest.mark.parametrize("N", [1, 2, 3, 5, 8, 9, 10, 256, 1000, 8192, 12289, 51201, 60001])      # <= 12288: 48 KB shared; <= 51200: opt-in shared; above: global
def test_permutation_bit_exact(N):
    for seed, epoch in [(1, 0), (1, 3), (2 ** 63 + 11, 7)]:
        got = host(binding.permutation(seed, epoch, N))
        assert np.array_equal(got, oracle.permutation(seed, epoch, N))
        assert np.array_equal(np.sort(got), np.arange(N))


# ---------------------------------------------------------------------------------------------------
# scans, distribution math, optimizer: fp32 kernels vs fp64 oracle
# ---------------------------------------------------------------------------------------------------
def _traj(T, B, seed, done_p=0.02):
    g = synth.rng(seed)
    V = g.standard_normal((T + 1, B)).astype(np.float32)
    r = g.choice(np.array([-1, 0, 1], np.float32), size=(T, B), p=[0.05, 0.9, 0.05]).astype(np.float32)
    d = (g.random((T, B)) < done_p).astype(np.uint8)
    logpi = (-np.abs(g.standard_normal((T, B))) - 1).astype(np.float32)
    logmu = (logpi + 0.3 * g.standard_normal((T, B))).astype(np.float32)
    return V, r, d, logpi, logmu


@pytest.mark.parametrize("T,B", [(20, 128), (5, 4), (1, 1), (128, 64), (20, 1000), (37, 131)])
@pytest.mark.parametrize("kw", [dict(), dict(lam=0.9, rho_bar=2.0, c_bar=1.5, rho_pg_bar=0.7), dict(gamma=1.0, c_bar=0.0)])
def test_vtrace_parity(T, B, kw):
    V, r, d, logpi, logmu = _traj(T, B, T * 1000 + B, done_p=0.1)
    vs, pg, rho = binding.vtrace(dev(V), dev(r), dev(d), dev(logpi), dev(logmu), **kw)
    rvs, rpg, rrho = oracle.vtrace(V, r, d, logpi, logmu, **kw)
    close(host(vs), rvs, 1e-5, what="vs"); close(host(pg), rpg, 1e-5, what="pgadv"); close(host(rho), rrho, 1e-5, what="rho")


@pytest.mark.parametrize("T,B", [(128, 64), (5, 4), (1, 1), (20, 1000), (37, 131)])
@pytest.mark.parametrize("lam", [0.95, 1.0, 0.0])
def test_gae_parity(T, B, lam):
    V, r, d, _, _ = _traj(T, B, T * 7 + B, done_p=0.1)
    adv, ret = binding.gae(dev(V), dev(r), dev(d), 0.99, lam)
    radv, rret = oracle.gae(V, r, d, 0.99, lam)
    close(host(adv), radv, 1e-5, what="adv"); close(host(ret), rret, 1e-5, what="ret")


def test_scans_all_dones_and_empty():
    T, B = 6, 40
    V, r, d, logpi, logmu = _traj(T, B, 5)
    d[:] = 1
    vs, pg, rho = binding.vtrace(dev(V), dev(r), dev(d), dev(logpi), dev(logmu))
    w = np.minimum(1.0, np.exp(logpi.astype(np.float64) - logmu))
    close(host(vs), V[:-1] + w * (r - V[:-1]), 1e-5, what="A1: all dones => vs = V + rho (r - V)")
    adv, _ = binding.gae(dev(V), dev(r), dev(d))
    close(host(adv), r.astype(np.float64) - V[:-1], 1e-5, what="A1: all dones => adv = r - V")
    e = torch.empty((0, 8), device="cuda"); e8 = torch.empty((0, 8), dtype=torch.uint8, device="cuda")
    binding.vtrace(torch.zeros((1, 8), device="cuda"), e, e8, e, e)   # T = 0: nothing to do, no error
    torch.cuda.synchronize()


def test_logprob_entropy_parity():
    g = synth.rng(3)
    logits = (g.standard_normal((1000, 18)) * 3).astype(np.float32); act = g.integers(0, 18, 1000).astype(np.int32)
    lp, H = binding.logprob_entropy(dev(logits), dev(act))
    rlp, rH = oracle.log_softmax(logits)
    close(host(lp), rlp[np.arange(1000), act], 1e-6, what="logp"); close(host(H), rH, 1e-6, what="entropy")


@pytest.mark.parametrize("P", [1, 3, 4, 4099, 100003, 1094115])
@pytest.mark.parametrize("k,gscale,max_norm", [(1, 1.0, 40.0), (100, 50.0, 0.5), (7, 1e-3, 40.0)])
def test_clip_adam_parity(P, k, gscale, max_norm):
    g = synth.rng(P + k)
    th = (g.standard_normal(P) * 0.05).astype(np.float32); grad = (g.standard_normal(P) * gscale / np.sqrt(P)).astype(np.float32)
    m = np.zeros(P, np.float32) if k == 1 else (g.standard_normal(P) * 0.01).astype(np.float32)
    v = np.zeros(P, np.float32) if k == 1 else (g.random(P) * 1e-4).astype(np.float32)
    dth, dm, dv = dev(th), dev(m), dev(v)
    gn = binding.clip_adam(dth, dm, dv, dev(grad), k, 6e-4, 0.9, 0.999, 1e-5, max_norm)
    rth, rm, rv, rn = oracle.clip_adam(th, m, v, grad.astype(np.float64), k, 6e-4, 0.9, float(np.float32(0.999)), 1e-5, max_norm)
    assert abs(float(host(gn)[0]) - rn) <= 1e-6 * rn
    close(host(dm), rm, 1e-5, what="m"); close(host(dv), rv, 1e-5, what="v")
    assert rel_l2(host(dth), rth) < 1e-6
    close(host(dth) - th, rth.astype(np.float64) - th, 1e-4, what="update")


def test_clip_adam_lr0_leaves_params_bit_identical():
    g = synth.rng(1); P = 5000
    th = g.standard_normal(P).astype(np.float32); dth = dev(th)
    binding.clip_adam(dth, dev(np.zeros(P, np.float32)), dev(np.zeros(P, np.float32)), dev(g.standard_normal(P).astype(np.float32)), 1, 0.0)
    assert host(dth).tobytes() == th.tobytes()


# ---------------------------------------------------------------------------------------------------
# losses with their adjoint seeds (a8), element by element: O5 (A4-A6) and O7 (Eq. 2-3, A5-A8)
# ---------------------------------------------------------------------------------------------------
def _loss_inputs(N, A, seed):
    g = synth.rng(seed)
    head = np.concatenate([g.standard_normal((N, A)) * 2.0, g.standard_normal((N, 1))], axis=1).astype(np.float32)
    act = g.integers(0, A, N).astype(np.int32)
    return g, head, act


@pytest.mark.parametrize("N,A", [(2560, 18), (1, 18), (131, 6), (20480, 18)])
@pytest.mark.parametrize("prec,red", [("fp32", 0), ("fp32", 1), ("bf16", 0)])
def test_impala_loss_seeds_parity(N, A, prec, red):
    g, head, act = _loss_inputs(N, A, N + A)
    vs = g.standard_normal(N).astype(np.float32); pg = g.standard_normal(N).astype(np.float32); rho = g.random(N).astype(np.float32)
    dhead, stats = binding.impala_loss(dev(head), dev(act), dev(vs), dev(pg), dev(rho), 0.5, 0.01, red, prec)
    st, dl, dV = oracle.impala_loss(head[:, :A], head[:, A], act, vs, pg, rho, 0.5, 0.01, red)
    got = host(dhead.float()); ref = np.concatenate([dl, dV[:, None]], axis=1)
    if prec == "fp32":
        close(got, ref, 1e-5, what="impala seeds")
    else:      # computed in fp32, stored as bf16: one rounding of relative size 2^-9
        assert (np.abs(got - ref) <= 2.0 ** -8 * np.abs(ref) + 1e-4 * np.sqrt(np.mean(ref ** 2))).all()
    gs = host(stats).astype(np.float64); scale = abs(st[1]) + abs(st[2]) + 1e-3
    tol = 1e-6 if prec == "fp32" else 2e-5
    for i in (0, 1, 2, 3, 7):
        assert abs(gs[i] - st[i]) <= tol * (abs(st[i]) + scale), (oracle.STAT_NAMES[i], gs[i], st[i])


@pytest.mark.parametrize("m,A,norm", [(2048, 18, 1), (2048, 18, 0), (3, 18, 1), (517, 6, 1)])
@pytest.mark.parametrize("prec", ["fp32", "bf16"])
def test_ppo_loss_seeds_parity(m, A, norm, prec):
    g, head, act_m = _loss_inputs(m, A, m + A + norm)
    N = 4 * m + 5                                                     # the minibatch gathers rows idx of the rollout arrays
    idx = g.permutation(N)[:m].astype(np.int32)
    act = g.integers(0, A, N).astype(np.int32); adv = g.standard_normal(N).astype(np.float32); ret = g.standard_normal(N).astype(np.float32)
    lp, _ = oracle.log_softmax(head[:, :A].astype(np.float64))
    lpo = np.zeros(N, np.float32); lpo[idx] = (lp[np.arange(m), act[idx]] + 0.15 * g.standard_normal(m)).astype(np.float32)      # ratios on both sides of the clip
    dhead, stats = binding.ppo_loss(dev(head), dev(idx), dev(act), dev(adv), dev(ret), dev(lpo), 0.1, 0.5, 0.01, norm, prec)
    st, dl, dV = oracle.ppo_loss(head[:, :A], head[:, A], act[idx], adv[idx], ret[idx], lpo[idx], 0.1, 0.5, 0.01, norm)
    assert m < 100 or 0.05 < st[6] < 0.95                              # clipped and unclipped samples both present
    got = host(dhead.float()); ref = np.concatenate([dl, dV[:, None]], axis=1)
    if prec == "fp32":
        close(got, ref, 1e-5, what="ppo seeds")
    else:
        # fp32 arithmetic: a ratio within 1e-6 of the clip boundary may fall on the other side (gradient switched off); none in this draw
        assert (np.abs(got - ref) <= 2.0 ** -8 * np.abs(ref) + 1e-4 * np.sqrt(np.mean(ref ** 2))).all()
    gs = host(stats).astype(np.float64); scale = abs(st[1]) + abs(st[2]) + 1e-3
    tol = 1e-6 if prec == "fp32" else 2e-5
    for i in (0, 1, 2, 3, 5, 6):
        assert abs(gs[i] - st[i]) <= tol * (abs(st[i]) + scale) + (1e-6 if i == 5 else 0), (oracle.STAT_NAMES[i], gs[i], st[i])
