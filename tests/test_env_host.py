"""CPU checks of the synthetic environment's numpy definition (synth.BlobEnv, the stand-in for EnvPool: PAPER.md:125, 166, 293) and of the
pipeline's host-side schedule arithmetic (Table 1)."""
import numpy as np

from paper_2310_00036_b200 import binding, build, synth


def test_blob_env_contract():
    arch = synth.ArchSpec("impala", (16, 32, 32), 256, 18, 4, 84, 84); B = 7
    env = synth.BlobEnv(B, 5, arch); o = env.reset()
    assert o.shape == (B, 4, 84, 84) and o.dtype == np.uint8 and (o[:, 0] == o[:, 3]).all()            # reset: the stack repeats one frame
    g = synth.rng(1); dones = 0; rewards = set()
    for step in range(400):
        prev = o
        o, r, d = env.step(g.integers(0, 18, B), step)
        assert r.dtype == np.float32 and d.dtype == np.uint8 and set(np.unique(r)) <= {-1.0, 0.0, 1.0}
        nd = d == 0
        assert (o[nd][:, :3] == prev[nd][:, 1:]).all()                                                 # stack shifts by one frame per step
        assert (o[~nd][:, 0] == o[~nd][:, 3]).all()                                                    # a done restarts the stack
        assert ((r == -1.0) <= (d == 1)).all()                                                         # the hazard ends the episode
        dones += int(d.sum()); rewards |= set(np.unique(r))
    assert 0.005 < dones / (400 * B) < 0.06 and o.max() > 100
    # a trajectory is a pure function of (seed, actions): replays agree, another seed does not
    a = synth.BlobEnv(3, 9, arch); b = synth.BlobEnv(3, 9, arch); c = synth.BlobEnv(3, 10, arch)
    oa, ob, oc = a.reset(), b.reset(), c.reset()
    assert np.array_equal(oa, ob) and not np.array_equal(oa, oc)
    for step in range(5):
        act = np.array([step % 18, 3, 17])
        assert all(np.array_equal(x, y) for x, y in zip(a.step(act, step), b.step(act, step)))


def test_hash_is_32_bit_and_spreads():
    h = synth.env_hash(2 ** 40 + 3, np.arange(4096), 7, 9)
    assert h.max() < 2 ** 32 and len(np.unique(h)) == 4096
    cnt = np.bincount((h % 16).astype(np.int64), minlength=16)
    assert ((cnt - 256.0) ** 2 / 256.0).sum() < 50.0                                                   # 15 dof


def test_policy_version_schedule_host():
    build.build()
    # Table 1: Synchronous pi_i; Cleanba pi_1, pi_1, pi_2, pi_3, ... (Figure 1 right: `if i != 2: params = param_Q.get()`)
    assert [binding.pipeline_policy_version(True, i) for i in range(1, 7)] == [1, 2, 3, 4, 5, 6]
    assert [binding.pipeline_policy_version(False, i) for i in range(1, 7)] == [1, 1, 2, 3, 4, 5]
    # the same schedule from a literal transcription of Figure 1's two loops with blocking queues of size 1
    import queue
    import threading
    import time
    for sync in (False, True):
        param_q, data_q, used, trained = queue.Queue(1), queue.Queue(1), [], []

        def actor():
            params = None
            for i in range(1, 7):
                if sync or i != 2:
                    params = param_q.get()
                used.append(params); data_q.put(params)            # the "data" is the version that collected it

        def learner():
            version = 1
            for _ in range(1, 7):
                data = data_q.get(); trained.append((data, version)); version += 1; param_q.put(version)

        param_q.put(1)
        ts = [threading.Thread(target=actor, daemon=True), threading.Thread(target=learner, daemon=True)]
        [t.start() for t in ts]
        ts[0].join(timeout=10)
        for _ in range(1000):                                      # the learner's last put() may block for ever (nobody is left to get): daemon thread
            if len(trained) == 6:
                break
            time.sleep(0.01)
        assert used == [binding.pipeline_policy_version(sync, i) for i in range(1, 7)]
        assert trained == [(binding.pipeline_policy_version(sync, i), i) for i in range(1, 7)]
