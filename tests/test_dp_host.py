"""Host logic of the data-parallel learner (paper_2310_00036_b200/dp.py) over a world_size-2 (and 3)
gloo group on CPU: the gradient exchange (all-to-all of rank chunks, rank-order sum, all-gather) returns the same bytes on every rank, equal
to the rank-ordered mean; with the ORACLE's shard gradients as inputs the exchanged gradient is the oracle's full-batch gradient
(App. A Option 1 = Option 2).  The sum is done here by a torch stand-in for cb_sum_ranks (its CUDA kernel is tested on the GPU in
tests/test_gpu_learner.py::test_sum_ranks_fixed_order); everything else is the product code."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _sum_ranks_cpu(slices, scale, out=None):
    import torch
    acc = slices[0].clone()
    for r in range(1, slices.shape[0]):
        acc += slices[r]                                  # rank order, fp32
    acc *= torch.tensor(scale, dtype=torch.float32)
    if out is not None:
        out.copy_(acc); return out
    return acc


def _worker(rank, world, port, P, q):
    import torch
    import torch.distributed as dist
    from paper_2310_00036_b200 import dp
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    g = torch.from_numpy(np.load(os.path.join(os.environ["DP_TEST_DIR"], f"g{rank}.npy")))
    ex = dp.GradientExchange(P, "cpu", sum_fn=_sum_ranks_cpu)
    out1 = ex(g.clone()).numpy().copy()
    out2 = ex(g.clone()).numpy().copy()                   # buffers are reused: a second exchange gives the same bytes
    dist.barrier(); dist.destroy_process_group()
    q.put((rank, out1.tobytes(), out2.tobytes()))


def _run(world, grads, port, tmp_path):
    import torch.multiprocessing as mp
    for r, g in enumerate(grads):
        np.save(tmp_path / f"g{r}.npy", g)
    os.environ["DP_TEST_DIR"] = str(tmp_path)
    ctx = mp.get_context("spawn"); q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, grads[0].size, q)) for r in range(world)]
    [p.start() for p in ps]
    out = sorted(q.get(timeout=180) for _ in ps)
    [p.join(60) for p in ps]
    assert all(p.exitcode == 0 for p in ps)
    return out


def test_exchange_world2_oracle_shard_gradients(tmp_path):
    from oracle import oracle as O
    from paper_2310_00036_b200 import dp, synth
    arch = synth.ArchSpec("impala", (2, 3, 3), 8, n_actions=5, in_c=2, in_h=13, in_w=13)
    oa = O.make_arch(arch.kind, arch.channels, arch.fc, arch.n_actions, arch.in_c, arch.in_h, arch.in_w)
    T, B = 3, 4
    rew, dones = synth.gen_rewards_dones(T, B, 2)
    obs = synth.gen_obs_uniform((T + 1) * B, 1, arch).reshape(T + 1, B, arch.in_c, arch.in_h, arch.in_w)
    bl, act = synth.gen_behaviour(T, B, arch.n_actions, 3)
    p = synth.gen_params(arch, 4, bias_scale=0.1).astype(np.float64)
    _, g_all = O.impala_objective_f64(oa, O.make_hparams("impala", T, B), p, p, obs, act, rew, dones, bl, want_grad=True)
    h2 = O.make_hparams("impala", T, B // 2); shards = []
    for s in (slice(0, 2), slice(2, 4)):
        _, gi = O.impala_objective_f64(oa, h2, p, p, obs[:, s], act[:, s], rew[:, s], dones[:, s], bl[:, s], want_grad=True)
        shards.append(gi.astype(np.float32))
    assert p.size % 2 == 1 or dp.chunk_elems(p.size, 2) * 2 > p.size          # the chunks are padded: the tail must not leak
    out = _run(2, shards, 29541, tmp_path)
    assert out[0][1] == out[1][1] == out[0][2] == out[1][2]                  # identical bytes on both ranks, and on a repeat
    got = np.frombuffer(out[0][1], np.float32)
    mean = ((shards[0] + shards[1]) * np.float32(0.5)).astype(np.float32)
    assert np.array_equal(got, mean)                                         # rank-order fp32 sum, then the scale
    np.testing.assert_allclose(got, g_all, rtol=2e-6, atol=1e-9)             # = the full-batch gradient


def test_exchange_world3_ragged(tmp_path):
    g = np.random.Generator(np.random.Philox(7))
    P = 1003                                                                  # not a multiple of 3 nor of 4
    grads = [(g.standard_normal(P) * 10.0 ** (3 * r)).astype(np.float32) for r in range(3)]
    out = _run(3, grads, 29551, tmp_path)
    assert out[0][1] == out[1][1] == out[2][1]
    acc = grads[0].copy()
    for r in (1, 2):
        acc = (acc + grads[r]).astype(np.float32)
    assert np.array_equal(np.frombuffer(out[0][1], np.float32), (acc * np.float32(1.0 / 3)).astype(np.float32))
