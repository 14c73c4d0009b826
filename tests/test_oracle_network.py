"""Pins for the oracle's network forward/backward (oracle O1, O2, O8; readings A10, A11).

Nothing here compares the oracle with itself: the references are torch-CPU fp64 library ops
(conv2d / max_pool2d / linear / autograd), brute-force window maxima, hand-built cases and
central finite differences.
"""
import numpy as np
import pytest
import torch
import torch.nn.functional as F

from oracle import oracle as O
from paper_2310_00036_b200 import synth

TINY_IMPALA = synth.ArchSpec("impala", (2, 3, 3), 8, n_actions=5, in_c=2, in_h=13, in_w=13)
TINY_NATURE = synth.ArchSpec("nature", (2, 3, 3), 8, n_actions=5, in_c=2, in_h=36, in_w=36)


def to_orc(a):
    return O.make_arch(a.kind, a.channels, a.fc, a.n_actions, a.in_c, a.in_h, a.in_w)


def split(arch, params):
    out, off = {}, 0
    for name, shape, _ in synth.param_tensors(arch):
        n = int(np.prod(shape)); out[name] = params[off:off + n].reshape(shape); off += n
    return out


def torch_pool_same(x):
    """3x3 s2 max-pool with XLA SAME padding built from library ops: pad with -inf then VALID pool."""
    H, W = x.shape[-2:]

    def pads(h):
        o = (h + 1) // 2; tot = max((o - 1) * 2 + 3 - h, 0); return tot // 2, tot - tot // 2
    (pt, pb), (pl, pr) = pads(H), pads(W)
    return F.max_pool2d(F.pad(x, (pl, pr, pt, pb), value=float("-inf")), 3, 2)


def torch_forward(arch, p, obs):
    """Independent restatement with torch library ops, fp64."""
    x = obs.double() / 255.0
    if arch.kind == "nature":
        x = F.relu(F.conv2d(x, p["conv1.w"], p["conv1.b"], stride=4))
        x = F.relu(F.conv2d(x, p["conv2.w"], p["conv2.b"], stride=2))
        x = F.relu(F.conv2d(x, p["conv3.w"], p["conv3.b"], stride=1))
    else:
        for s in range(3):
            x = F.conv2d(x, p[f"stage{s}.conv.w"], p[f"stage{s}.conv.b"], padding=1)
            x = torch_pool_same(x)
            for b in range(2):
                h = F.conv2d(F.relu(x), p[f"stage{s}.block{b}.conv1.w"], p[f"stage{s}.block{b}.conv1.b"], padding=1)
                h = F.conv2d(F.relu(h), p[f"stage{s}.block{b}.conv2.w"], p[f"stage{s}.block{b}.conv2.b"], padding=1)
                x = x + h
        x = F.relu(x)
    h = F.relu(F.linear(x.flatten(1), p["fc.w"], p["fc.b"]))
    return F.linear(h, p["pi.w"], p["pi.b"]), F.linear(h, p["v.w"], p["v.b"])[:, 0]


def torch_params(arch, params, grad=False):
    return {k: torch.tensor(v, dtype=torch.float64, requires_grad=grad) for k, v in split(arch, params).items()}


def test_param_counts_and_layout():
    # 1 693 875 / 1 094 115 / 4 364 211 parameters
    for arch, n in ((synth.NATURE, 1693875), (synth.IMPALA, 1094115), (synth.IMPALA_WIDE, 4364211)):
        assert synth.param_count(arch) == n
        assert O.param_count(to_orc(arch)) == n
        off = 0
        for (name, shape, fan), (o_off, o_cnt, o_fan) in zip(synth.param_tensors(arch), O.param_tensors(to_orc(arch))):
            assert (off, int(np.prod(shape)), fan) == (o_off, o_cnt, o_fan), name
            off += int(np.prod(shape))
    assert O.feature_shape(to_orc(synth.IMPALA)) == (32, 11, 11)      # 84 -> 42 -> 21 -> 11 (A10)
    assert O.feature_shape(to_orc(synth.NATURE)) == (64, 7, 7)        # 84 -> 20 -> 9 -> 7


@pytest.mark.parametrize("arch", [TINY_IMPALA, TINY_NATURE, synth.IMPALA, synth.NATURE])
def test_forward_matches_torch_library_ops(arch):
    params = synth.gen_params(arch, 7, bias_scale=0.1)
    nf = 3 if arch.in_h < 84 else 2
    obs = synth.gen_obs_uniform(nf, 11, arch)
    lg, v = O.forward(to_orc(arch), params, obs)
    tl, tv = torch_forward(arch, torch_params(arch, params), torch.from_numpy(obs))
    np.testing.assert_allclose(lg, tl.numpy(), rtol=1e-10, atol=1e-11)
    np.testing.assert_allclose(v, tv.numpy(), rtol=1e-10, atol=1e-11)
    lg32, v32 = O.forward_f32(to_orc(arch), params, obs)
    assert lg32.dtype == np.float32 and np.array_equal(lg32, lg.astype(np.float32)) and np.array_equal(v32, v.astype(np.float32))


@pytest.mark.parametrize("arch", [TINY_IMPALA, TINY_NATURE])
def test_backward_matches_torch_autograd(arch):
    params = synth.gen_params(arch, 3, bias_scale=0.1)
    obs = synth.gen_obs_uniform(4, 5, arch)
    g = synth.rng(9); dl = g.standard_normal((4, arch.n_actions)); dv = g.standard_normal(4)
    grad = O.backward_f64(to_orc(arch), params.astype(np.float64), obs, dl, dv)
    tp = torch_params(arch, params, grad=True)
    tl, tv = torch_forward(arch, tp, torch.from_numpy(obs))
    ((tl * torch.from_numpy(dl)).sum() + (tv * torch.from_numpy(dv)).sum()).backward()
    ref = np.concatenate([tp[name].grad.numpy().ravel() for name, _, _ in synth.param_tensors(arch)])
    np.testing.assert_allclose(grad, ref, rtol=1e-9, atol=1e-12)


def test_backward_full_size_impala_one_frame_vs_autograd():
    arch = synth.IMPALA
    params = synth.gen_params(arch, 21, bias_scale=0.05)
    obs = synth.gen_obs_blobs(1, 1, 4, arch)[0]
    g = synth.rng(2); dl = g.standard_normal((1, 18)); dv = g.standard_normal(1)
    grad = O.backward_f64(to_orc(arch), params.astype(np.float64), obs, dl, dv)
    tp = torch_params(arch, params, grad=True)
    tl, tv = torch_forward(arch, tp, torch.from_numpy(obs))
    ((tl * torch.from_numpy(dl)).sum() + (tv * torch.from_numpy(dv)).sum()).backward()
    ref = np.concatenate([tp[name].grad.numpy().ravel() for name, _, _ in synth.param_tensors(arch)])
    np.testing.assert_allclose(grad, ref, rtol=1e-8, atol=1e-11)


@pytest.mark.parametrize("arch", [TINY_IMPALA, TINY_NATURE])
def test_backward_brute_force_finite_differences(arch):
    """central differences in fp64, h = 1e-6 max(1,|theta|), every parameter of the tiny net."""
    oa = to_orc(arch)
    p = synth.gen_params(arch, 13, bias_scale=0.1).astype(np.float64)
    obs = synth.gen_obs_uniform(2, 17, arch)
    g = synth.rng(1); dl = g.standard_normal((2, arch.n_actions)); dv = g.standard_normal(2)

    def f(q):
        lg, v = O.forward_f64(oa, q, obs); return float((lg * dl).sum() + (v * dv).sum())
    grad = O.backward_f64(oa, p, obs, dl, dv)
    idx = np.arange(p.size) if p.size <= 1500 else synth.rng(3).choice(p.size, 1500, replace=False)
    fd = np.empty(idx.size)
    for n, i in enumerate(idx):
        h = 1e-6 * max(1.0, abs(p[i])); q = p.copy(); q[i] += h; up = f(q); q[i] -= 2 * h; fd[n] = (up - f(q)) / (2 * h)
    scale = np.abs(grad).max()
    assert np.abs(fd - grad[idx]).max() <= 2e-6 * scale


def test_maxpool_same_padding_shapes_and_brute_force():
    for h, pads in ((84, (0, 1)), (42, (0, 1)), (21, (1, 1)), (11, (1, 1)), (13, (1, 1)), (7, (1, 1))):
        o = (h + 1) // 2; tot = max((o - 1) * 2 + 3 - h, 0)
        assert (tot // 2, tot - tot // 2) == pads                      # A10 worked values
        x = synth.rng(h).standard_normal((2, h, h))
        y, arg = O.maxpool_same(x)
        assert y.shape == (2, o, o)
        xp = np.full((2, h + tot, h + tot), -np.inf); xp[:, pads[0]:pads[0] + h, pads[0]:pads[0] + h] = x
        for c in range(2):
            for i in range(o):
                for j in range(o):
                    assert y[c, i, j] == xp[c, 2 * i:2 * i + 3, 2 * j:2 * j + 3].max()
                    assert x.ravel()[arg[c, i, j]] == y[c, i, j]
        np.testing.assert_array_equal(y, torch_pool_same(torch.from_numpy(x)[None])[0].numpy())


def test_maxpool_constant_ramp_and_tie_rule():
    y, arg = O.maxpool_same(np.full((1, 6, 6), 2.5))
    assert np.all(y == 2.5)
    # tie -> FIRST element of the window in row-major order (A11); 6x6, pads (0,1): window (i,j) starts at (2i,2j)
    assert arg[0, 0, 0] == 0 and arg[0, 1, 1] == 2 * 6 + 2 and arg[0, 2, 2] == 4 * 6 + 4
    ramp = np.arange(49, dtype=np.float64).reshape(1, 7, 7)              # strictly increasing: last in-range wins
    y, arg = O.maxpool_same(ramp)                                         # 7 -> 4, pads (1,1)
    assert y[0, 0, 0] == ramp[0, 1, 1] and y[0, 3, 3] == ramp[0, 6, 6] and arg[0, 3, 3] == 48
    # hand-built tie: two equal maxima in one window, gradient must go to the first one only
    x = np.zeros((1, 5, 5)); x[0, 1, 2] = 9.0; x[0, 2, 1] = 9.0
    y, arg = O.maxpool_same(x)                                            # 5 -> 3, pads (1,1); window(1,1) rows 1..3, cols 1..3
    assert y[0, 1, 1] == 9.0 and arg[0, 1, 1] == 1 * 5 + 2


def test_softmax_entropy_identities():
    g = synth.rng(5); lg = g.standard_normal((64, 18)) * 3
    lp, H = O.log_softmax(lg)
    np.testing.assert_allclose(np.exp(lp).sum(1), 1.0, rtol=1e-14)
    np.testing.assert_allclose(lp - lp[:, :1], lg - lg[:, :1], rtol=1e-12, atol=1e-12)      # log p_i - log p_0 = l_i - l_0
    lp2, H2 = O.log_softmax(lg + 123.25)                                                    # shift invariance
    np.testing.assert_allclose(lp2, lp, atol=1e-12); np.testing.assert_allclose(H2, H, atol=1e-12)
    lpu, Hu = O.log_softmax(np.zeros((1, 18)))
    np.testing.assert_allclose(Hu, np.log(18.0), rtol=1e-14); np.testing.assert_allclose(lpu, -np.log(18.0), rtol=1e-14)
    lpd, Hd = O.log_softmax(np.array([[50.0] + [0.0] * 17]))                                # near-deterministic: H -> 0
    assert 0 <= Hd[0] < 1e-17
    np.testing.assert_allclose(H, torch.distributions.Categorical(logits=torch.from_numpy(lg)).entropy().numpy(), rtol=1e-12)
