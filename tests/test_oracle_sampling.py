"""Pins for the oracle's counter-based sampler (oracle O3; reading A9).

Philox4x32-10 is pinned to cuRAND's HOST generator (a library implementation that runs without a
GPU); the fixed-operation log to libm over every uniform the sampler can produce; the sampler as
a whole to its distribution (chi-square against softmax) and to invariances.
"""
import ctypes as C
import glob
import os

import numpy as np
import pytest

from oracle import oracle as O
from paper_2310_00036_b200 import synth


def _curand():
    for pat in ("/usr/local/cuda/lib64/libcurand.so*", "/usr/local/cuda*/targets/*/lib/libcurand.so*"):
        for p in sorted(glob.glob(pat)):
            try:
                return C.CDLL(p)
            except OSError:
                pass
    try:
        import nvidia.curand  # pip wheel layout
        for p in glob.glob(os.path.join(os.path.dirname(nvidia.curand.__file__), "lib", "libcurand.so*")):
            return C.CDLL(p)
    except Exception:
        pass
    return None


def _curand_host_stream(seed, n):
    cr = _curand()
    if cr is None:
        pytest.skip("libcurand not found")
    gen = C.c_void_p()
    assert cr.curandCreateGeneratorHost(C.byref(gen), C.c_int(161)) == 0          # CURAND_RNG_PSEUDO_PHILOX4_32_10
    assert cr.curandSetPseudoRandomGeneratorSeed(gen, C.c_ulonglong(seed)) == 0
    out = np.empty(n, np.uint32)
    assert cr.curandGenerate(gen, out.ctypes.data_as(C.c_void_p), C.c_size_t(n)) == 0
    cr.curandDestroyGenerator(gen)
    return out


@pytest.mark.parametrize("seed", [0, 0x0123456789ABCDEF, 2 ** 64 - 1])
def test_philox_matches_curand_host_generator(seed):
    n = 1 << 20
    ref = _curand_host_stream(seed, n).reshape(-1, 4)
    key = [seed & 0xFFFFFFFF, seed >> 32]
    # cuRAND's host ordering: block i of the stream is Philox(counter = (r, 0, s, 0), key = seed) with
    # i = r * S + s for some number S of interleaved subsequences; discover S from the stream itself.
    first_r1 = O.philox([1, 0, 0, 0], key)
    hits = np.nonzero((ref == first_r1).all(1))[0]
    assert hits.size == 1, "counter (1,0,0,0) not found in the library stream"
    S = int(hits[0])
    idx = np.arange(ref.shape[0])
    mine = np.array([O.philox([i // S, 0, i % S, 0], key) for i in idx[:: max(1, ref.shape[0] // 250000)]])
    assert np.array_equal(mine, ref[:: max(1, ref.shape[0] // 250000)])


def test_philox_counter_and_key_words_all_matter():
    base = O.philox([1, 2, 3, 4], [5, 6])
    for w in range(4):
        c = [1, 2, 3, 4]; c[w] ^= 1
        assert not np.array_equal(O.philox(c, [5, 6]), base)
    assert not np.array_equal(O.philox([1, 2, 3, 4], [4, 6]), base)
    assert not np.array_equal(O.philox([1, 2, 3, 4], [5, 7]), base)


def test_fixed_log_within_2ulp_of_libm_on_every_uniform():
    worst = 0.0
    for lo in range(0, 1 << 24, 1 << 20):
        u = (np.arange(lo, lo + (1 << 20), dtype=np.float64) + 0.5) * 2.0 ** -24
        mine = O.fixed_log_u24(lo, 1 << 20); ref = np.log(u)
        worst = max(worst, float(np.max(np.abs(mine - ref) / np.spacing(np.abs(ref)))))
    assert worst <= 2.0, worst
    # second application: arguments -log(u) in (2.9e-8, 17.4)
    x = -np.log((synth.rng(1).integers(0, 1 << 24, 200000) + 0.5) * 2.0 ** -24)
    mine = np.array([O.fixed_log(v) for v in x[:20000]])
    assert np.max(np.abs(mine - np.log(x[:20000])) / np.spacing(np.abs(np.log(x[:20000])) + 1e-300)) <= 4.0
    for v in (1.0, 2.0, 0.5, 1.4142135623730951, 1e-7, 17.0):
        assert abs(O.fixed_log(v) - np.log(v)) <= 2 * np.spacing(abs(np.log(v)) + 1e-300) + 1e-17


def test_gumbel_table_is_fp32_rounding_of_the_definition():
    lo, n = 0, 1 << 16
    for lo in (0, 1 << 12, (1 << 24) - (1 << 16)):
        g = O.gumbel_table(lo, n)
        u = (np.arange(lo, lo + n, dtype=np.float64) + 0.5) * 2.0 ** -24
        ref = -np.log(-np.log(u))
        assert g.dtype == np.float32
        assert np.max(np.abs(g.astype(np.float64) - ref) / np.spacing(np.abs(ref).astype(np.float32)).astype(np.float64)) <= 0.5001 + 1e-3
    assert np.isfinite(O.gumbel_table(0, 1)).all() and np.isfinite(O.gumbel_table((1 << 24) - 1, 1)).all()


def test_sampler_distribution_chi_square():
    A, n = 18, 1_000_000
    logits = (synth.rng(7).standard_normal(A) * 1.5).astype(np.float32)
    acts = O.sample(np.tile(logits, (n, 1)), seed=99, step=3, env_offset=0)
    p = np.exp(logits.astype(np.float64) - logits.max()); p /= p.sum()
    cnt = np.bincount(acts, minlength=A)
    chi2 = ((cnt - n * p) ** 2 / (n * p)).sum()
    assert chi2 < 50.0, chi2                                              # 17 dof: P(chi2 > 50) ~ 4e-5


def test_sampler_invariances_and_keys():
    g = synth.rng(3); lg = g.standard_normal((4096, 18)).astype(np.float32)
    lg = np.round(lg * 64) / 64                                           # exactly representable shifts below
    a = O.sample(lg, seed=5, step=9, env_offset=100)
    assert np.array_equal(a, O.sample(lg + np.float32(8.0), seed=5, step=9, env_offset=100))      # shift invariance
    assert np.array_equal(a, O.sample(lg, seed=5, step=9, env_offset=100))                        # deterministic
    assert not np.array_equal(a, O.sample(lg, seed=6, step=9, env_offset=100))
    assert not np.array_equal(a, O.sample(lg, seed=5, step=10, env_offset=100))
    assert not np.array_equal(a, O.sample(lg, seed=5, step=9, env_offset=101))
    assert np.array_equal(a[7:], O.sample(lg[7:], seed=5, step=9, env_offset=107))                # keyed by env id
    big = lg.copy(); big[:, 11] += 1000.0
    assert np.all(O.sample(big, seed=1, step=1) == 11)                                            # dominant logit
    assert np.all(O.sample(np.full((64, 18), -np.inf, np.float32), 1, 1) == 0)                    # all-ties -> lowest index
    # independent restatement with libm log: mismatches only where the top-2 scores are a near-tie
    key = [5, 0]
    ref = np.empty(256, np.int32)
    for b in range(256):
        w = np.concatenate([O.philox([100 + b, 9, 0, j], key) for j in range(5)])[:18]
        u = ((w >> 8).astype(np.float64) + 0.5) * 2.0 ** -24
        sc = lg[b] + (-np.log(-np.log(u))).astype(np.float32)
        ref[b] = int(np.argmax(sc))
    assert np.array_equal(ref, a[:256])
