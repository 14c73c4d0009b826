"""CPU-side checks of the C-ABI library: it loads without a GPU, exports every symbol that
include/cleanba.h declares, and its host logic (layer table, parameter layout, cb_net_init,
argument validation) is right.  No compute call is made here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from oracle import oracle
from paper_2310_00036_b200 import binding, build, synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    build.build()


def _orc_arch(a):
    return oracle.make_arch(a.kind, a.channels, a.fc, a.n_actions, a.in_c, a.in_h, a.in_w)


def test_header_symbols_exported():
    hdr = open(os.path.join(ROOT, "include", "cleanba.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = sorted(set(re.findall(r"\b(cb_[a-z0-9_]+)\s*\(", hdr)))
    assert len(names) >= 15
    lib = binding.lib()
    for n in names:
        assert hasattr(lib, n), f"{n} declared in cleanba.h but not exported"
    assert sorted(binding.EXPORTS) == names


@pytest.mark.parametrize("arch", [synth.NATURE, synth.IMPALA, synth.IMPALA_WIDE,
                                  synth.ArchSpec("impala", (3, 5, 7), 11, 6, 2, 20, 23)])
def test_param_layout_matches_oracle_and_synth(arch):
    net = binding.Net(arch)
    lay = net.param_layout()
    exp = synth.param_tensors(arch)
    assert [n for n, _, _ in lay] == [n for n, _, _ in exp]
    assert [tuple(d) for _, _, d in lay] == [tuple(s) for _, s, _ in exp]
    offs = np.cumsum([0] + [int(np.prod(s)) for _, s, _ in exp])
    assert [o for _, o, _ in lay] == list(offs[:-1])
    assert net.P == offs[-1] == oracle.param_count(_orc_arch(arch))
    assert [o for o, _, _ in oracle.param_tensors(_orc_arch(arch))] == list(offs[:-1])


def test_published_param_counts():
    # SURVEY.md section 8 table (derived from BASELINE.json's shapes)
    assert binding.Net(synth.NATURE).P == 1693875
    assert binding.Net(synth.IMPALA).P == 1094115
    assert binding.Net(synth.IMPALA_WIDE).P == 4364211


def test_net_init_he_normal():
    net = binding.Net(synth.IMPALA)
    p1, p2, p3 = net.init_params(7), net.init_params(7), net.init_params(8)
    assert p1.tobytes() == p2.tobytes() and p1.tobytes() != p3.tobytes()
    for (name, off, dims), (_, _, fan) in zip(net.param_layout(), synth.param_tensors(synth.IMPALA)):
        n = int(np.prod(dims)); x = p1[off:off + n].astype(np.float64)
        if name.endswith(".b"):
            assert not x.any()
            continue
        sd = np.sqrt(2.0 / fan)
        assert abs(x.mean()) < 4 * sd / np.sqrt(n)
        if n >= 500:   # chi-square spread of the sample variance: rel. sd = sqrt(2/n)
            assert abs(x.var() / sd ** 2 - 1) < 4 * np.sqrt(2.0 / n) + 1e-3


def test_bad_arguments_are_errors_not_crashes():
    lib = binding.lib()
    h = C.c_void_p()
    a = binding.CArch(); a.kind = 7
    assert lib.cb_net_create(C.byref(a), 0, C.byref(h)) == -1 and not h
    assert b"arch" in lib.cb_last_error()
    assert lib.cb_net_create(None, 0, C.byref(h)) == -1
    net = binding.Net(synth.NATURE)
    assert lib.cb_param_layout(net._h, 999, None, None, None, None) == -1
    assert lib.cb_policy_forward(net._h, None, None, 4, 0, 0, 0, 0, None, None, None, None) == -1
    assert lib.cb_learner_step(net._h, None, None, None, None, None, None, None, None, None, None, None, None, None) == -1
    assert lib.cb_learner_grad(net._h, 0, None, None) == -1 and lib.cb_learner_apply(net._h, 0, None) == -1      # no cb_learner_begin
    with pytest.raises(binding.CleanbaError):
        binding.Net(synth.ArchSpec("nature", (32, 64, 64), 512, 18, 4, 20, 20))


def test_hparams_defaults_are_the_papers_tables():
    # Table 2 and Table 3
    p = binding.make_hparams("ppo"); i = binding.make_hparams("impala")
    assert (p.gamma, p.lambda_, p.clip_eps) == pytest.approx((0.99, 0.95, 0.1))
    assert (p.epochs, p.minibatches, p.norm_adv) == (4, 4, 1)
    assert (p.vf_coef, p.ent_coef, p.max_grad_norm, p.lr, p.adam_eps) == pytest.approx((0.5, 0.01, 0.5, 2.5e-4, 1e-5))
    assert (i.rho_bar, i.c_bar, i.lambda_, i.vf_coef, i.ent_coef, i.max_grad_norm) == pytest.approx((1, 1, 1, 0.5, 0.01, 40.0))
    o = oracle.make_hparams("ppo")
    for f in ("gamma", "lambda_", "clip_eps", "vf_coef", "ent_coef", "lr", "max_grad_norm", "adam_eps", "beta1", "beta2"):
        assert getattr(o, f) == pytest.approx(getattr(p, f))


def test_batch_bookkeeping_worked_example():
    # 8 envs x 128 steps = 1024, 4 minibatches of 256, K = 4 epochs -> 16 updates
    hp = binding.make_hparams("ppo", T=128, B=8)
    assert hp.T * hp.B == 1024 and hp.T * hp.B // hp.minibatches == 256 and hp.epochs * hp.minibatches == 16


def test_impala_defaults_and_linear_lr_host():
    i = binding.make_hparams("impala")
    assert i.minibatches == 1 and i.optimizer == 0 and (i.rms_decay, i.rms_eps) == pytest.approx((0.99, 0.01))     # Table 3
    # cb_linear_lr is host arithmetic: compare with the oracle's closed form
    for k, total in [(0, 100), (25, 100), (100, 100), (500, 100), (3, 0)]:
        assert binding.linear_lr(6e-4, k, total) == pytest.approx(oracle.linear_lr(float(np.float32(6e-4)), k, total), rel=1e-6, abs=1e-12)
