"""Pins for the oracle's V-trace, GAE, losses, clip+Adam, permutation and learner step
(oracle O4-O7, O9; readings A1-A8, A12, A13, A17).  References: brute-force double loops,
closed forms, invariants and finite differences -- never the oracle's own formula retyped.
"""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2310_00036_b200 import synth

TINY = synth.ArchSpec("impala", (2, 3, 3), 8, n_actions=5, in_c=2, in_h=13, in_w=13)


def to_orc(a):
    return O.make_arch(a.kind, a.channels, a.fc, a.n_actions, a.in_c, a.in_h, a.in_w)


def traj(T, B, seed, p_done=0.15):
    g = synth.rng(seed)
    V = g.standard_normal((T + 1, B)); r = g.standard_normal((T, B)); d = (g.random((T, B)) < p_done).astype(np.uint8)
    logpi = -np.abs(g.standard_normal((T, B))); logmu = logpi + 0.5 * g.standard_normal((T, B))
    return V, r, d, logpi, logmu


def brute_nstep_return(V, r, d, gamma):
    """G_t = sum_{k>=t} (prod_{j=t}^{k-1} disc_j) r_k + (prod_{j=t}^{T-1} disc_j) V_T, disc = gamma(1-d)."""
    T, B = r.shape; G = np.zeros((T, B))
    for b in range(B):
        for t in range(T):
            acc, prod = 0.0, 1.0
            for k in range(t, T):
                acc += prod * r[k, b]; prod *= gamma * (1.0 - d[k, b])
            G[t, b] = acc + prod * V[T, b]
    return G


# ------------------------------------------------------------------ V-trace (A2) -----------------
def test_vtrace_on_policy_equals_nstep_return():
    V, r, d, logpi, _ = traj(11, 5, 1)
    vs, pg, rho = O.vtrace(V, r, d, logpi, logpi)                       # w == 1, rho_bar = c_bar = lambda = 1
    G = brute_nstep_return(V, r, d, 0.99)
    np.testing.assert_allclose(vs, G, rtol=1e-12, atol=1e-12)
    np.testing.assert_allclose(rho, 1.0)
    # (iv) pgadv = r + disc vs_{t+1} - V_t  == GAE(lambda=1) advantage
    adv, _ = O.gae(V, r, d, 0.99, 1.0)
    np.testing.assert_allclose(pg, adv, rtol=1e-12, atol=1e-12)


def test_vtrace_cbar_zero_and_T1():
    V, r, d, logpi, logmu = traj(9, 4, 2)
    vs, pg, rho = O.vtrace(V, r, d, logpi, logmu, c_bar=0.0)
    w = np.exp(logpi - logmu); disc = 0.99 * (1.0 - d)
    np.testing.assert_allclose(vs, V[:-1] + np.minimum(1.0, w) * (r + disc * V[1:] - V[:-1]), rtol=1e-12, atol=1e-13)
    V, r, d, logpi, logmu = traj(1, 6, 3)
    vs, pg, rho = O.vtrace(V, r, d, logpi, logmu, rho_bar=1e30, c_bar=1e30, rho_pg_bar=1e30)
    w = np.exp(logpi - logmu); disc = 0.99 * (1.0 - d)
    np.testing.assert_allclose(vs[0], V[0] + w[0] * (r[0] + disc[0] * V[1] - V[0]), rtol=1e-12)
    np.testing.assert_allclose(pg[0], w[0] * (r[0] + disc[0] * V[1] - V[0]), rtol=1e-12)


@pytest.mark.parametrize("lam", [0.0, 0.3, 0.95, 1.0])
def test_vtrace_lambda_cross_pins_gae(lam):
    V, r, d, logpi, _ = traj(13, 3, 4)
    vs, pg, _ = O.vtrace(V, r, d, logpi, logpi, lam=lam)
    adv, ret = O.gae(V, r, d, 0.99, lam)
    np.testing.assert_allclose(vs - V[:-1], adv, rtol=1e-11, atol=1e-12)          # (iii)
    np.testing.assert_allclose(ret - V[:-1], adv, rtol=0, atol=1e-13)             # R - V = A identically (A3)


def test_done_cuts_dependence_and_all_done_case():
    V, r, d, logpi, logmu = traj(10, 2, 5, p_done=0.0)
    d[4, :] = 1
    a = O.vtrace(V, r, d, logpi, logmu); g1 = O.gae(V, r, d)
    V2, r2 = V.copy(), r.copy(); V2[5:] += 7.0; r2[5:] -= 3.0; lp2 = logpi.copy(); lp2[5:] -= 0.7
    b = O.vtrace(V2, r2, d, lp2, logmu); g2 = O.gae(V2, r2, d)
    assert np.array_equal(a[0][:5], b[0][:5]) and np.array_equal(a[1][:5], b[1][:5])        # A1: bit-identical
    assert np.array_equal(g1[0][:5], g2[0][:5])
    d[:] = 1
    vs, pg, rho = O.vtrace(V, r, d, logpi, logmu); adv, _ = O.gae(V, r, d)
    np.testing.assert_allclose(vs, V[:-1] + rho * (r - V[:-1]), rtol=1e-13)
    np.testing.assert_allclose(adv, r - V[:-1], rtol=1e-13)


def test_vtrace_clipping_thresholds():
    V, r, d, logpi, logmu = traj(6, 64, 6)
    _, _, rho = O.vtrace(V, r, d, logpi, logmu, rho_bar=0.8)
    w = np.exp(logpi - logmu)
    assert (w > 0.8).any() and (w < 0.8).any()
    np.testing.assert_allclose(rho, np.minimum(0.8, w), rtol=1e-14)


def brute_vtrace_definition(V, r, d, w, gamma, lam, rho_bar, c_bar):
    """Espeholt et al. 2018, Eq. 1, written out as the explicit double sum (no recursion):
    vs_t = V_t + sum_{k>=t} (prod_{j=t}^{k-1} disc_j c_j) rho_k (r_k + disc_k V_{k+1} - V_k), c_j = lam min(c_bar, w_j)."""
    T, B = r.shape; vs = np.zeros((T, B))
    for b in range(B):
        for t in range(T):
            acc, prod = 0.0, 1.0
            for k in range(t, T):
                disc = gamma * (1.0 - d[k, b])
                acc += prod * min(rho_bar, w[k, b]) * (r[k, b] + disc * V[k + 1, b] - V[k, b])
                prod *= disc * lam * min(c_bar, w[k, b])
            vs[t, b] = V[t, b] + acc
    return vs


@pytest.mark.parametrize("lam", [0.3, 0.95])
def test_vtrace_pgadv_lambda_mix_on_policy(lam):
    """The lambda mix inside q_t (A2): on-policy, q_t - V_t = delta_t + disc_t lam (vs_{t+1} - V_{t+1}), and with w == 1 the
    bracket is the GAE(lam) advantage at t+1, so pgadv_t is the GAE(lam) advantage at t -- computed here as the explicit
    double sum of discounted TD errors.  A q_t that used vs_{t+1} alone (lam = 1) or V_{t+1} alone would fail."""
    T, B, gam = 12, 4, 0.99
    V, r, d, logpi, _ = traj(T, B, 21)
    _, pg, _ = O.vtrace(V, r, d, logpi, logpi, gamma=gam, lam=lam)
    delta = r + gam * (1.0 - d) * V[1:] - V[:-1]
    ref = np.zeros((T, B))
    for b in range(B):
        for t in range(T):
            prod = 1.0
            for k in range(t, T):
                ref[t, b] += prod * delta[k, b]; prod *= gam * lam * (1.0 - d[k, b])
    np.testing.assert_allclose(pg, ref, rtol=1e-11, atol=1e-12)
    # the two degenerate mixes differ from it by far more than the tolerance (so the pin can fail)
    _, pg1, _ = O.vtrace(V, r, d, logpi, logpi, gamma=gam, lam=1.0)
    assert np.abs(pg1 - ref).max() > 1e-3 and np.abs(delta - ref).max() > 1e-3


def test_vtrace_off_policy_definition_and_separate_pg_threshold():
    """General off-policy case against the definition as a double sum, with three DIFFERENT thresholds (rho_bar = 2,
    c_bar = 1.5, rho_pg_bar = 0.7) and lam = 0.9: pgadv = min(rho_pg_bar, w) (r + disc (lam vs_{t+1} + (1-lam) V_{t+1}) - V)."""
    T, B, gam, lam = 10, 16, 0.99, 0.9
    V, r, d, logpi, logmu = traj(T, B, 22)
    w = np.exp(logpi - logmu)
    assert (w > 2.0).any() and ((w > 0.7) & (w < 1.5)).any() and ((w > 1.5) & (w < 2.0)).any() and (w < 0.7).any()
    vs, pg, rho = O.vtrace(V, r, d, logpi, logmu, gamma=gam, lam=lam, rho_bar=2.0, c_bar=1.5, rho_pg_bar=0.7)
    vs_ref = brute_vtrace_definition(V, r, d, w, gam, lam, 2.0, 1.5)
    np.testing.assert_allclose(vs, vs_ref, rtol=1e-11, atol=1e-12)
    vs_next = np.concatenate([vs_ref[1:], V[-1:]], axis=0)                        # vs_T = V_T
    q = r + gam * (1.0 - d) * (lam * vs_next + (1.0 - lam) * V[1:])
    pg_ref = np.minimum(0.7, w) * (q - V[:-1])
    np.testing.assert_allclose(pg, pg_ref, rtol=1e-11, atol=1e-12)
    np.testing.assert_allclose(rho, np.minimum(2.0, w), rtol=1e-14)
    # a pgadv clipped at rho_bar instead of rho_pg_bar would be visibly different
    assert np.abs(np.minimum(2.0, w) * (q - V[:-1]) - pg_ref).max() > 1e-2


# ------------------------------------------------------------------ GAE (A3) ---------------------
def test_gae_lambda_one_and_zero():
    V, r, d, _, _ = traj(17, 4, 7)
    adv, ret = O.gae(V, r, d, 0.97, 1.0)
    np.testing.assert_allclose(adv, brute_nstep_return(V, r, d, 0.97) - V[:-1], rtol=1e-12, atol=1e-12)
    adv0, _ = O.gae(V, r, d, 0.97, 0.0)
    np.testing.assert_allclose(adv0, r + 0.97 * (1.0 - d) * V[1:] - V[:-1], rtol=1e-14)


def test_gae_brute_force_general_lambda():
    V, r, d, _, _ = traj(9, 3, 8); gam, lam = 0.99, 0.95
    adv, _ = O.gae(V, r, d, gam, lam)
    delta = r + gam * (1.0 - d) * V[1:] - V[:-1]
    ref = np.zeros_like(adv)
    for b in range(3):
        for t in range(9):
            prod = 1.0
            for k in range(t, 9):
                ref[t, b] += prod * delta[k, b]; prod *= gam * lam * (1.0 - d[k, b])
    np.testing.assert_allclose(adv, ref, rtol=1e-12, atol=1e-13)


# ------------------------------------------------------------------ losses -----------------------
def rand_batch(N, A, seed):
    g = synth.rng(seed)
    return (g.standard_normal((N, A)), g.standard_normal(N), g.integers(0, A, N).astype(np.int32),
            g.standard_normal(N), g.standard_normal(N))


def test_impala_loss_seeds_by_finite_differences_and_reduction_linearity():
    N, A = 7, 5; lg, V, act, vs, pg = rand_batch(N, A, 1)
    st, dl, dV = O.impala_loss(lg, V, act, vs, pg, c1=0.5, c2=0.01)
    h = 1e-6
    for n in range(N):
        for i in range(A):
            p = lg.copy(); p[n, i] += h; m = lg.copy(); m[n, i] -= h
            fd = (O.impala_loss(p, V, act, vs, pg)[0][0] - O.impala_loss(m, V, act, vs, pg)[0][0]) / (2 * h)
            assert abs(fd - dl[n, i]) < 1e-8
        p = V.copy(); p[n] += h; m = V.copy(); m[n] -= h
        fd = (O.impala_loss(lg, p, act, vs, pg)[0][0] - O.impala_loss(lg, m, act, vs, pg)[0][0]) / (2 * h)
        assert abs(fd - dV[n]) < 1e-8
    st1, dl1, dV1 = O.impala_loss(lg, V, act, vs, pg, reduction=1)                       # A4: sum = N x mean
    np.testing.assert_allclose(dl1, N * dl, rtol=1e-13); np.testing.assert_allclose(dV1, N * dV, rtol=1e-13)
    np.testing.assert_allclose(st1[0], N * st[0], rtol=1e-12)
    # A5: value-only derivative, dL/dV_n = -c1 (vs - V)/N ; sign tests (A6)
    np.testing.assert_allclose(dV, -0.5 * (vs - V) / N, rtol=1e-13)
    assert O.impala_loss(lg * 0.0, V, act, vs, pg)[0][3] > st[3]                           # uniform policy has max entropy
    lo = O.impala_loss(lg, V, act, vs, pg, c2=0.0)[0][0]; hi = O.impala_loss(lg, V, act, vs, pg, c2=1.0)[0][0]
    np.testing.assert_allclose(lo - hi, st[3], rtol=1e-12)                                 # more entropy weight lowers L by H
    np.testing.assert_allclose(st[0], st[1] + 0.5 * st[2] - 0.01 * st[3], rtol=1e-13)


def test_ppo_ratio_one_invariants():
    m, A = 64, 6; lg, V, act, adv, ret = rand_batch(m, A, 2)
    lp, H = O.log_softmax(lg); lpo = lp[np.arange(m), act]
    st, dl, dV = O.ppo_loss(lg, V, act, adv, ret, lpo, eps=0.1)
    assert st[5] == 0.0 and st[6] == 0.0                                    # approx_kl = 0, clip_frac = 0 exactly
    At = (adv - adv.mean()) / (adv.std() + 1e-8)
    np.testing.assert_allclose(st[1], -At.mean(), atol=1e-15)               # L_pg = -mean(Atil) ~ 0
    assert abs(st[1]) < 1e-15
    # gradient of L_pg at ratio 1 = gradient of the vanilla policy-gradient surrogate -mean(Atil log pi)
    p = np.exp(lp); onehot = np.eye(A)[act]
    vanilla = -(At[:, None] * (onehot - p)) / m
    ent = 0.01 * p * (lp + H[:, None]) / m
    np.testing.assert_allclose(dl, vanilla + ent, rtol=1e-10, atol=1e-15)
    np.testing.assert_allclose(dV, 0.5 * (V - ret) / m, rtol=1e-13)


def test_ppo_clipping_and_finite_differences():
    m, A = 48, 5; lg, V, act, adv, ret = rand_batch(m, A, 3)
    lp, _ = O.log_softmax(lg); g = synth.rng(4)
    lpo = lp[np.arange(m), act] + 0.25 * g.standard_normal(m)               # ratios spread around 1 +- 0.25
    st, dl, dV = O.ppo_loss(lg, V, act, adv, ret, lpo, eps=0.1)
    r = np.exp(lp[np.arange(m), act] - lpo)
    np.testing.assert_allclose(st[6], (np.abs(r - 1) > 0.1).mean(), rtol=1e-14)
    np.testing.assert_allclose(st[5], ((r - 1) - np.log(r)).mean(), rtol=1e-12)
    assert 0 < st[6] < 1
    h = 1e-6
    for n in range(0, m, 5):
        for i in range(A):
            a = lg.copy(); a[n, i] += h; b = lg.copy(); b[n, i] -= h
            fd = (O.ppo_loss(a, V, act, adv, ret, lpo)[0][0] - O.ppo_loss(b, V, act, adv, ret, lpo)[0][0]) / (2 * h)
            assert abs(fd - dl[n, i]) < 1e-8
    # Eq. 2 by brute force: J = mean min(r A, clip(r) A)
    At = (adv - adv.mean()) / (adv.std() + 1e-8)
    J = np.minimum(r * At, np.clip(r, 0.9, 1.1) * At).mean()
    np.testing.assert_allclose(st[1], -J, rtol=1e-12)


def test_advantage_normalisation_properties():
    m, A = 256, 4; lg, V, act, adv, ret = rand_batch(m, A, 5)
    lp, _ = O.log_softmax(lg); lpo = lp[np.arange(m), act] + 0.05
    a = O.ppo_loss(lg, V, act, adv, ret, lpo)[1]
    b = O.ppo_loss(lg, V, act, 37.0 * adv + 5.0, ret, lpo)[1]               # A8: invariant to affine rescaling (k > 0)
    np.testing.assert_allclose(a, b, rtol=1e-6, atol=1e-12)
    c = O.ppo_loss(lg, V, act, adv, ret, lpo, norm_adv=0)[1]
    assert not np.allclose(a, c)


# ------------------------------------------------------------------ clip + Adam (A12, A13) -------
def test_adam_first_step_closed_form_and_lr_zero():
    g64 = synth.rng(1).standard_normal(1000) * 0.01; th = synth.rng(2).standard_normal(1000).astype(np.float32)
    z = np.zeros(1000, np.float32)
    th1, m1, v1, n = O.clip_adam(th, z, z, g64, 1, lr=6e-4, eps=1e-5, max_norm=40.0)
    np.testing.assert_allclose(n, np.sqrt((g64 ** 2).sum()), rtol=1e-14)
    expect = th.astype(np.float64) - 6e-4 * g64 / (np.abs(g64) + 1e-5)       # first step from zero state
    np.testing.assert_allclose(th1, expect.astype(np.float32), rtol=0, atol=1e-7 * 1.0)
    th0, _, _, _ = O.clip_adam(th, z, z, g64, 1, lr=0.0)
    assert np.array_equal(th0, th)


def test_adam_constant_gradient_and_clip():
    P = 64; g64 = synth.rng(3).standard_normal(P); th = np.zeros(P, np.float32); m = np.zeros(P, np.float32); v = m.copy()
    c = 0.5; n0 = np.sqrt((g64 ** 2).sum()); gc = g64 * c / n0               # A13: post-clip norm = min(n, c)
    for k in range(1, 6):
        th, m, v, n = O.clip_adam(th, m, v, g64, k, lr=1e-3, eps=1e-5, max_norm=c)
        np.testing.assert_allclose(m / (1 - 0.9 ** k), gc, rtol=2e-6)        # m_hat = g, v_hat = g^2 at every k
        np.testing.assert_allclose(v / (1 - 0.999 ** k), gc ** 2, rtol=2e-6)
    # scaling the gradient by 10 when ||g|| > c leaves the update unchanged
    z = np.zeros(P, np.float32)
    a = O.clip_adam(z, z, z, g64, 1, lr=1e-3, max_norm=c)[0]; b = O.clip_adam(z, z, z, 10 * g64, 1, lr=1e-3, max_norm=c)[0]
    np.testing.assert_allclose(a, b, rtol=1e-6)
    # identity when ||g|| <= c
    small = g64 * 0.01
    a = O.clip_adam(z, z, z, small, 1, lr=1e-3, max_norm=1e9)[1]; b = O.clip_adam(z, z, z, small, 1, lr=1e-3, max_norm=n0 * 0.01 * 1.0001)[1]
    assert np.array_equal(a, b)


# ------------------------------------------------------------------ permutation (A17) ------------
def test_permutation_is_a_bijection_and_follows_the_index_rule():
    for N in (1, 2, 5, 1024, 8192):
        p = O.permutation(123, 2, N)
        assert np.array_equal(np.sort(p), np.arange(N))
    assert not np.array_equal(O.permutation(123, 0, 1024), O.permutation(123, 1, 1024))
    assert not np.array_equal(O.permutation(123, 0, 1024), O.permutation(124, 0, 1024))
    assert np.array_equal(O.permutation(123, 3, 1024), O.permutation(123, 3, 1024))
    # brute-force restatement of the rule from Philox words only
    N, seed, epoch = 37, 0xABCDEF0123, 1
    words = np.concatenate([O.philox([q, epoch, 0, 0x5045524D], [seed & 0xFFFFFFFF, seed >> 32]) for q in range(10)])
    ref = list(range(N))
    for q, i in enumerate(range(N - 1, 0, -1)):
        j = (int(words[q]) * (i + 1)) >> 32; ref[i], ref[j] = ref[j], ref[i]
    assert list(O.permutation(seed, epoch, N)) == ref
    # uniformity smoke: position of element 0 over many seeds ~ uniform
    pos = np.array([int(np.nonzero(O.permutation(s, 0, 8) == 0)[0][0]) for s in range(4000)])
    cnt = np.bincount(pos, minlength=8); chi2 = ((cnt - 500.0) ** 2 / 500.0).sum()
    assert chi2 < 30.0                                                       # 7 dof, p ~ 1e-4


# ------------------------------------------------------------------ whole learner step -----------
def make_step_inputs(T, B, seed, arch=TINY):
    g = synth.rng(seed); A = arch.n_actions
    obs = synth.gen_obs_uniform((T + 1) * B, seed, arch)
    bl = g.standard_normal((T, B, A)).astype(np.float32)
    act = synth.categorical_from_uniform(bl, g.random((T, B)))
    rew, dones = synth.gen_rewards_dones(T, B, seed + 1)
    return obs, act, rew, dones, bl


def test_impala_objective_gradient_by_finite_differences_targets_constant():
    arch = TINY; oa = to_orc(arch); T, B = 3, 2
    obs, act, rew, dones, bl = make_step_inputs(T, B, 31)
    hp = O.make_hparams("impala", T, B)
    p = synth.gen_params(arch, 5, bias_scale=0.1).astype(np.float64)
    L, grad = O.impala_objective_f64(oa, hp, p, p, obs, act, rew, dones, bl, want_grad=True)
    idx = synth.rng(6).choice(p.size, 300, replace=False)
    for i in idx:
        h = 1e-6 * max(1.0, abs(p[i])); q = p.copy(); q[i] += h
        up = O.impala_objective_f64(oa, hp, q, p, obs, act, rew, dones, bl); q[i] -= 2 * h
        fd = (up - O.impala_objective_f64(oa, hp, q, p, obs, act, rew, dones, bl)) / (2 * h)
        assert abs(fd - grad[i]) <= 1e-6 * max(np.abs(grad).max(), 1e-3), i
    # the learner step reports the same loss and uses the same gradient
    p32 = p.astype(np.float32); z = np.zeros_like(p32)
    out = O.learner_step(oa, hp, p32, z, z, 0, obs, act, rew, dones, bl, debug=True)
    L32, g32 = O.impala_objective_f64(oa, hp, p32.astype(np.float64), p32.astype(np.float64), obs, act, rew, dones, bl, want_grad=True)
    np.testing.assert_allclose(out["stats"][0, 0], L32, rtol=1e-6)
    np.testing.assert_allclose(out["grad"], g32, rtol=1e-12, atol=1e-15)
    np.testing.assert_allclose(out["stats"][0, 4], np.sqrt((g32 ** 2).sum()), rtol=1e-6)
    assert out["opt_step"] == 1
    exp_p, _, _, _ = O.clip_adam(p32, z, z, g32, 1, hp.lr, hp.beta1, hp.beta2, hp.adam_eps, hp.max_grad_norm)
    assert np.array_equal(out["params"], exp_p)


def test_ppo_objective_gradient_by_finite_differences():
    arch = TINY; oa = to_orc(arch); m = 6
    g = synth.rng(8); obs = synth.gen_obs_uniform(m, 41, arch)
    act = g.integers(0, arch.n_actions, m).astype(np.int32); adv = g.standard_normal(m); ret = g.standard_normal(m)
    p = synth.gen_params(arch, 9, bias_scale=0.1).astype(np.float64)
    lg, _ = O.forward_f64(oa, p, obs); lp, _ = O.log_softmax(lg)
    lpo = lp[np.arange(m), act] + 0.08 * g.standard_normal(m)
    hp = O.make_hparams("ppo", 3, 2)
    L, grad = O.ppo_objective_f64(oa, hp, p, obs, act, adv, ret, lpo, want_grad=True)
    for i in synth.rng(10).choice(p.size, 300, replace=False):
        h = 1e-6 * max(1.0, abs(p[i])); q = p.copy(); q[i] += h
        up = O.ppo_objective_f64(oa, hp, q, obs, act, adv, ret, lpo); q[i] -= 2 * h
        fd = (up - O.ppo_objective_f64(oa, hp, q, obs, act, adv, ret, lpo)) / (2 * h)
        assert abs(fd - grad[i]) <= 1e-6 * max(np.abs(grad).max(), 1e-3), i


def test_ppo_step_bookkeeping_and_single_minibatch_reduction():
    """App. A worked example scaled down: N = T*B samples, 4 minibatches x K=4 epochs -> 16 updates."""
    arch = TINY; oa = to_orc(arch); T, B = 4, 4
    obs, act, rew, dones, bl = make_step_inputs(T, B, 51)
    p = synth.gen_params(arch, 11, bias_scale=0.1); z = np.zeros_like(p)
    hp = O.make_hparams("ppo", T, B, epochs=4, minibatches=4)
    out = O.learner_step(oa, hp, p, z, z, 0, obs, act, rew, dones, bl)
    assert out["stats"].shape == (16, 8) and out["opt_step"] == 16
    assert np.isfinite(out["stats"]).all() and not np.array_equal(out["params"], p)
    # epochs = minibatches = 1: one full-batch update whose loss is permutation-invariant (A17)
    hp1 = O.make_hparams("ppo", T, B, epochs=1, minibatches=1)
    o1 = O.learner_step(oa, hp1, p, z, z, 0, obs, act, rew, dones, bl, debug=True)
    lg, V = o1["logits"][:T * B], o1["values"]
    adv, ret = O.gae(V.reshape(T + 1, B), rew, dones, 0.99, 0.95)
    np.testing.assert_allclose(o1["t0"], adv.ravel(), rtol=1e-13); np.testing.assert_allclose(o1["t1"], ret.ravel(), rtol=1e-13)
    lpb, _ = O.log_softmax(bl.reshape(T * B, -1).astype(np.float64)); lpo = lpb[np.arange(T * B), act.ravel()]
    st, _, _ = O.ppo_loss(lg, V[:T * B], act.ravel(), adv.ravel(), ret.ravel(), lpo)
    np.testing.assert_allclose(o1["stats"][0, :4], st[:4], rtol=2e-6, atol=1e-7)
    assert o1["opt_step"] == 1


def test_data_parallel_gradient_identity():
    """App. A Option 1 vs Option 2: gradient over B envs = mean of the gradients of env shards."""
    arch = TINY; oa = to_orc(arch); T, B = 3, 4
    obs, act, rew, dones, bl = make_step_inputs(T, B, 61)
    obs = obs.reshape(T + 1, B, *obs.shape[1:]); p = synth.gen_params(arch, 12, bias_scale=0.1).astype(np.float64)
    hp = O.make_hparams("impala", T, B)
    _, g_all = O.impala_objective_f64(oa, hp, p, p, obs, act, rew, dones, bl, want_grad=True)
    hp2 = O.make_hparams("impala", T, B // 2); gs = []
    for s in (slice(0, 2), slice(2, 4)):
        _, gi = O.impala_objective_f64(oa, hp2, p, p, obs[:, s], act[:, s], rew[:, s], dones[:, s], bl[:, s], want_grad=True)
        gs.append(gi)
    np.testing.assert_allclose(g_all, 0.5 * (gs[0] + gs[1]), rtol=1e-10, atol=1e-14)


# ---------------------------------------------------------------------------------------------------
# NEXT row f1: RMSprop (A22), env-split IMPALA minibatches (A21), linear LR anneal
# ---------------------------------------------------------------------------------------------------
def test_rmsprop_first_step_and_constant_gradient_closed_forms():
    g = synth.rng(5).standard_normal(300) * 0.01
    th0 = np.zeros(300, np.float32) + 0.5
    lr, d, eps = 6e-4, 0.99, 0.01
    th, nu, n = O.clip_rmsprop(th0, np.zeros(300, np.float32), g, lr, d, eps, max_norm=40.0)
    assert n == pytest.approx(np.linalg.norm(g), rel=1e-12)
    np.testing.assert_allclose(th.astype(np.float64) - 0.5, -lr * g / np.sqrt((1 - d) * g * g + eps), rtol=0, atol=1e-7)
    np.testing.assert_allclose(nu, (1 - d) * g * g, rtol=1e-6)
    # constant gradient for k steps: nu_k = (1 - d^k) g^2
    th, nu = th0, np.zeros(300, np.float32)
    for k in range(1, 6):
        th, nu, _ = O.clip_rmsprop(th, nu, g, lr, d, eps, 40.0)
        np.testing.assert_allclose(nu, (1 - d ** k) * g * g, rtol=2e-6)
    # lr = 0 leaves the parameters bit-identical; above the clip threshold the update ignores the gradient's scale
    th_z, _, _ = O.clip_rmsprop(th0, np.zeros(300, np.float32), g, 0.0, d, eps, 40.0)
    assert th_z.tobytes() == th0.tobytes()
    a, _, _ = O.clip_rmsprop(th0, np.zeros(300, np.float32), g * 1e3, lr, d, eps, 0.5)
    b, _, _ = O.clip_rmsprop(th0, np.zeros(300, np.float32), g * 1e4, lr, d, eps, 0.5)
    np.testing.assert_allclose(a, b, rtol=0, atol=1e-7)


def test_linear_lr_anneal():
    # Tables 2-3 "linear decay to 0"
    assert O.linear_lr(6e-4, 0, 100) == 6e-4 and O.linear_lr(6e-4, 100, 100) == 0.0
    assert O.linear_lr(6e-4, 25, 100) == pytest.approx(4.5e-4, rel=1e-12) and O.linear_lr(6e-4, 500, 100) == 0.0


def test_impala_env_split_minibatches_equal_sequential_single_steps():
    """A21: mb env-groups = mb full learner steps on the groups, in order, with the parameters flowing."""
    arch = synth.ArchSpec("impala", (3, 4, 5), 12, 5, 2, 20, 20)
    oa = O.make_arch(arch.kind, arch.channels, arch.fc, arch.n_actions, arch.in_c, arch.in_h, arch.in_w)
    T, B, mb = 3, 6, 3
    rewards, dones = synth.gen_rewards_dones(T, B, 1)
    obs = synth.gen_obs_uniform((T + 1) * B, 2, arch).reshape(T + 1, B, arch.in_c, arch.in_h, arch.in_w)
    bl, act = synth.gen_behaviour(T, B, arch.n_actions, 3)
    p0 = synth.gen_params(arch, 4, bias_scale=0.05); P = p0.size
    for opt in (0, 1):
        hp = O.make_hparams("impala", T, B, minibatches=mb, optimizer=opt)
        out = O.learner_step(oa, hp, p0, np.zeros(P, np.float32), np.zeros(P, np.float32), 0, obs, act, rewards, dones, bl)
        assert out["stats"].shape[0] == mb and out["opt_step"] == mb
        p, m, v, k = p0, np.zeros(P, np.float32), np.zeros(P, np.float32), 0
        Bm = B // mb
        for g in range(mb):
            sl = slice(g * Bm, (g + 1) * Bm)
            h1 = O.make_hparams("impala", T, Bm, minibatches=1, optimizer=opt)
            o1 = O.learner_step(oa, h1, p, m, v, k, np.ascontiguousarray(obs[:, sl]), np.ascontiguousarray(act[:, sl]),
                                     np.ascontiguousarray(rewards[:, sl]), np.ascontiguousarray(dones[:, sl]), np.ascontiguousarray(bl[:, sl]))
            p, m, v, k = o1["params"], o1["m"], o1["v"], o1["opt_step"]
            np.testing.assert_array_equal(out["stats"][g], o1["stats"][0])
        assert out["params"].tobytes() == p.tobytes() and out["v"].tobytes() == v.tobytes()
        if opt == 1:
            assert not out["m"].any()          # RMSprop keeps its state in the second buffer only


# ---------------------------------------------------------------------------------------------------
# NEXT row f4: actor-time values for GAE (A3b, Alg. 1 l.8-12), the epoch
# counter of the PPO permutation (A23) and RMSprop under the PPO schedule
# ---------------------------------------------------------------------------------------------------
def _ppo_by_hand(oa, hp, p, m, v, k, obs, act, rew, dones, bl, values, epoch0):
    """Alg. 1 l.11-20 composed from the separately pinned pieces: GAE on `values`, per-epoch permutation, and for every
    minibatch the PPO objective gradient (finite-difference-pinned) followed by clip + Adam (closed-form-pinned)."""
    T, B = hp.T, hp.B; N = T * B; A = bl.shape[-1]
    adv, ret = O.gae(values.reshape(T + 1, B).astype(np.float64), rew, dones, hp.gamma, hp.lambda_)
    lpb, _ = O.log_softmax(bl.reshape(N, A).astype(np.float64)); lpo = lpb[np.arange(N), act.ravel()]
    frames = obs.reshape((T + 1) * B, *obs.shape[-3:]); mbs = N // hp.minibatches; losses = []
    for e in range(hp.epochs):
        perm = O.permutation(hp.perm_seed, epoch0 + e, N)
        for j in range(hp.minibatches):
            idx = perm[j * mbs:(j + 1) * mbs]
            L, g = O.ppo_objective_f64(oa, hp, p.astype(np.float64), frames[idx], act.ravel()[idx], adv.ravel()[idx], ret.ravel()[idx], lpo[idx], want_grad=True)
            k += 1
            p, m, v, _ = O.clip_adam(p, m, v, g, k, hp.lr, hp.beta1, hp.beta2, hp.adam_eps, hp.max_grad_norm)
            losses.append(L)
    return p, m, v, k, np.array(losses), adv, ret


def test_ppo_behaviour_values_and_epoch_counter():
    arch = TINY; oa = to_orc(arch); T, B = 4, 3
    obs, act, rew, dones, bl = make_step_inputs(T, B, 71)
    p = synth.gen_params(arch, 13, bias_scale=0.1); z = np.zeros_like(p)
    hp = O.make_hparams("ppo", T, B, epochs=2, minibatches=2, perm_seed=9)
    # (1) NULL = recompute (A3): equals the hand composition on the oracle's own fp64 values
    o0 = O.learner_step(oa, hp, p, z, z, 0, obs, act, rew, dones, bl, debug=True)
    ph, mh, vh, kh, Lh, adv, ret = _ppo_by_hand(oa, hp, p, z, z, 0, obs, act, rew, dones, bl, o0["values"], 0)
    assert o0["params"].tobytes() == ph.tobytes() and o0["m"].tobytes() == mh.tobytes() and o0["v"].tobytes() == vh.tobytes() and kh == 4
    np.testing.assert_allclose(o0["stats"][:, 0], Lh, rtol=2e-6, atol=1e-7)
    # (2) actor-time values = the same values as the ABI carries them (fp32): bit-identical to the hand composition on
    #     those fp32 values, and within fp32 rounding of the recomputing step
    bv = o0["values"].astype(np.float32)
    o1 = O.learner_step(oa, hp, p, z, z, 0, obs, act, rew, dones, bl, debug=True, behaviour_values=bv)
    ph, mh, vh, _, Lh, adv, ret = _ppo_by_hand(oa, hp, p, z, z, 0, obs, act, rew, dones, bl, bv, 0)
    assert o1["params"].tobytes() == ph.tobytes() and o1["v"].tobytes() == vh.tobytes()
    np.testing.assert_array_equal(o1["t0"], adv.ravel()); np.testing.assert_array_equal(o1["t1"], ret.ravel())
    np.testing.assert_allclose(o1["t0"], o0["t0"], rtol=0, atol=1e-5)
    # (3) values of ANOTHER policy (what the Cleanba architecture hands the learner: D of the second latest policy) change the
    #     targets, and only through GAE: the step still equals the hand composition
    bv2 = (bv + synth.rng(72).standard_normal(bv.size).astype(np.float32) * 0.3).astype(np.float32)
    o2 = O.learner_step(oa, hp, p, z, z, 0, obs, act, rew, dones, bl, debug=True, behaviour_values=bv2)
    ph, _, _, _, _, adv2, _ = _ppo_by_hand(oa, hp, p, z, z, 0, obs, act, rew, dones, bl, bv2, 0)
    assert o2["params"].tobytes() == ph.tobytes() and np.abs(adv2 - adv).max() > 1e-2
    # IMPALA ignores the argument (V-trace uses the current parameters' values, O4)
    hi = O.make_hparams("impala", T, B)
    a = O.learner_step(oa, hi, p, z, z, 0, obs, act, rew, dones, bl); b = O.learner_step(oa, hi, p, z, z, 0, obs, act, rew, dones, bl, behaviour_values=bv2)
    assert a["params"].tobytes() == b["params"].tobytes()
    # (4) A23: a call entered with opt_step = 4 (= after one call of 2 x 2 updates) continues with epochs 2, 3
    o3 = O.learner_step(oa, hp, o0["params"], o0["m"], o0["v"], 4, obs, act, rew, dones, bl, debug=True)
    ph, _, _, kh, _, _, _ = _ppo_by_hand(oa, hp, o0["params"], o0["m"], o0["v"], 4, obs, act, rew, dones, bl, o3["values"], 2)
    assert o3["params"].tobytes() == ph.tobytes() and o3["opt_step"] == kh == 8
    assert not np.array_equal(O.permutation(9, 2, T * B), O.permutation(9, 0, T * B))


def test_ppo_with_rmsprop_follows_the_same_schedule():
    """cb_hparams.optimizer = 1 under the PPO schedule (reachable through the ABI): each update is clip + RMSprop (A22)."""
    arch = TINY; oa = to_orc(arch); T, B = 3, 2
    obs, act, rew, dones, bl = make_step_inputs(T, B, 81)
    p = synth.gen_params(arch, 14, bias_scale=0.1); z = np.zeros_like(p)
    hp = O.make_hparams("ppo", T, B, epochs=1, minibatches=1, optimizer=1)
    o = O.learner_step(oa, hp, p, z, z, 0, obs, act, rew, dones, bl, debug=True)
    th, nu, n = O.clip_rmsprop(p, z, o["grad"], hp.lr, hp.rms_decay, hp.rms_eps, hp.max_grad_norm)
    assert o["params"].tobytes() == th.tobytes() and o["v"].tobytes() == nu.tobytes() and not o["m"].any()
    assert o["stats"][0, 4] == pytest.approx(n, rel=1e-6)
