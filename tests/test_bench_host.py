"""Host logic of bench.py: the N > 1 aggregation (max of per-rank times, sum of per-rank frames) over a
world_size-2 gloo group on CPU, the workload bookkeeping and the reference arm's JSON contract."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, q):
    import torch.distributed as dist
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    t = bench.max_over_ranks(1.0 + rank, world)          # rank 1 is the slow one
    f = bench.sum_over_ranks(2560.0 * 10, world)
    dist.barrier(); dist.destroy_process_group()
    q.put((rank, t, f))


def test_aggregation_world2_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn"); q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, 29531, q)) for r in range(2)]
    [p.start() for p in ps]
    out = sorted(q.get(timeout=120) for _ in ps)
    [p.join(60) for p in ps]
    assert all(p.exitcode == 0 for p in ps)
    for rank, t, f in out:
        assert t == 2.0 and f == 51200.0      # whole-job frames / max-over-ranks time
    import bench
    assert bench.max_over_ranks(3.5, 1) == 3.5


def test_useful_flops_match_survey_table():
    import bench
    from paper_2310_00036_b200 import synth
    # 826 G (config 2), 11.29 T (config 3), 25.75 T (config 4)
    assert bench.useful_flops_per_step(synth.CONFIGS[2]) == pytest.approx(826e9, rel=2e-3)
    assert bench.useful_flops_per_step(synth.CONFIGS[3]) == pytest.approx(11.29e12, rel=2e-3)
    assert bench.useful_flops_per_step(synth.CONFIGS[4]) == pytest.approx(25.75e12, rel=2e-3)


def test_reference_arm_json_contract():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0", "--config", "0"],
                         capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "env-frames/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    # non-zero ranks of a torchrun launch exit 0 without work
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"], capture_output=True, text=True, timeout=60, cwd=ROOT, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""
