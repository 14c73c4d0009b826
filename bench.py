#!/usr/bin/env python
"""bench.py -- learner env-frames/s of the Cleanba hot path on B200 (BASELINE.json's metric).

A "step" is one cb_learner_step (forward over (T+1)B frames, V-trace or GAE, loss, backward, global
clip + Adam) over one batch of seeded synthetic trajectories shaped like the paper's Atari runs.
Default workload: BASELINE.json configs[2] (IMPALA-ResNet 16/32/32, T=20, B=128, bf16 mode), the
configuration the learner metric is quoted on; --config 3 / 4 select the PPO and the wide workloads.
N > 1 (torchrun): N independent replicas, one per GPU, no data-path collective ("replicas only",
DESIGN.md section 7) -- weak scaling; with --dp the N ranks form ONE data-parallel learner instead (B envs per rank, one
fixed-order gradient exchange per update: paper_2310_00036_b200/dp.py).  `--impl reference` times the CPU oracle instead.
The default line also carries: per-step median / min, `other_configs` (configs 3 and 4, a few steps each), `hbm_kernels`
(scan / loss / norm / optimizer kernels against the HBM roof at the BASELINE shapes and at a scaled-up shape), `pipeline`
(Cleanba's actor/learner architecture against the Synchronous one) and `inference` (configs[1]).

Prints ONE JSON line (rank 0).  See DESIGN.md section 6 for every key.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2310_00036_b200 import synth  # noqa: E402

METRIC = "learner env-frames/sec on 1 B200 (fwd+V-trace/GAE+bwd+Adam); % bf16 TC peak"
UNIT = "env-frames/s"
# useful MACs per frame: forward, backward (dgrad + wgrad, no dgrad into obs)
MACS = {"impala": (54_227_712, 104_391_168), "impala_wide": (208_772_608, 409_416_704), "nature": (9_352_704, 15_428_608)}
N_ROTATE = 3      # distinct input sets cycled through so that observations are never L2-resident


def workload(cfg_index):
    cfg = synth.CONFIGS[cfg_index]
    if cfg["algo"] == "actor":
        raise SystemExit("config 1 is actor inference only; the learner metric is quoted on configs 2-4")
    return cfg


def net_key(arch):
    return "nature" if arch.kind == "nature" else ("impala_wide" if arch.channels[0] == 32 else "impala")


def useful_flops_per_step(cfg):
    f, b = MACS[net_key(cfg["arch"])]
    T, B = cfg["T"], cfg["B"]
    if cfg["algo"] == "ppo":      # one no-grad forward over (T+1)B frames + epochs x (forward + backward) over T*B
        return 2.0 * (f * (T + 1) * B + 4 * (f + b) * T * B)
    return 2.0 * (f * (T + 1) * B + b * T * B)


def gen_inputs(cfg_index, cfg, n_sets, rank):
    """n_sets seeded input sets (host numpy).  Behaviour logits ~ N(0,1) for config 0, else N(0, 0.3) around
    a fixed seeded logit field (the bench does not need the policy-coupled recipe A18: throughput does not
    depend on the values)."""
    T, B, arch = cfg["T"], cfg["B"], cfg["arch"]
    sets = []
    for i in range(n_sets):
        seed = 1000 + cfg_index + 7919 * i + 104729 * rank
        rewards, dones = synth.gen_rewards_dones(T, B, seed + 1)
        if cfg["obs"] == "uniform":
            obs = synth.gen_obs_uniform((T + 1) * B, seed, arch).reshape(T + 1, B, arch.in_c, arch.in_h, arch.in_w)
        else:
            # blobs for a slice of envs, tiled to B envs with a per-copy horizontal shift (np.roll): same statistics, bounded generation time
            nb = min(B, 32)
            base = synth.gen_obs_blobs(T + 1, nb, seed, arch, dones[:, :nb])
            reps = (B + nb - 1) // nb
            obs = np.concatenate([np.roll(base, r * 3, axis=-1) for r in range(reps)], axis=1)[:, :B]
        bl, actions = synth.gen_behaviour(T, B, arch.n_actions, seed + 2, None, 0.3)
        sets.append(dict(obs=np.ascontiguousarray(obs), actions=actions, rewards=rewards, dones=dones, behaviour_logits=bl))
    return sets


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 50 ms.  The process is started BEFORE the warm-up steps (nvidia-smi
    needs a few hundred ms to come up, longer than a short timed region); a reader thread stamps every sample with its arrival
    time and stop() keeps the samples that fall between begin() and end(), i.e. during the timed region."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, gpu_index):
        self.p = None; self.lines = []; self.t0 = self.t1 = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "50"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True, bufsize=1)
        except OSError:
            return
        import threading

        def reader():
            for line in self.p.stdout:
                self.lines.append((time.perf_counter(), line))
        self.th = threading.Thread(target=reader, daemon=True); self.th.start()

    def begin(self):
        self.t0 = time.perf_counter()

    def end(self):
        self.t1 = time.perf_counter()

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.06)      # let the sample in flight arrive
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.th.join(timeout=2)
        t0 = self.t0 if self.t0 is not None else 0.0; t1 = (self.t1 if self.t1 is not None else time.perf_counter()) + 0.06
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, line in self.lines:
            if not (t0 <= ts <= t1):
                continue
            f = [x.strip() for x in line.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": sorted(reasons), "samples": len(sm)}


def max_over_ranks(t_local, world):
    """Max of a per-rank scalar over all ranks (identity for world == 1).  Works with nccl and gloo."""
    if world == 1:
        return t_local
    import torch
    import torch.distributed as dist
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([t_local], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x_local, world):
    if world == 1:
        return x_local
    import torch
    import torch.distributed as dist
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([x_local], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def pick_tensor_peak(peaks, clk):
    """The bf16 roof that fits the run: the burst figure when the SM clock sat at its maximum for the whole timed region (no power cap),
    the sustained figure otherwise (MEASURED_PEAKS.json took it at a ~1.3 GHz median)."""
    at_max = clk.get("sm_mhz") and clk.get("sm_max_mhz") and clk["sm_mhz"] >= 0.97 * clk["sm_max_mhz"] and "sw_power_cap" not in clk.get("reasons", [])
    if at_max:
        return peaks["tf_burst"], f"{peaks['src']} (burst bf16: SM clock at max during the timed region)"
    return peaks["tf_sust"], f"{peaks['src']} (sustained bf16: SM clock below max or power-capped during the timed region)"


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=d["hbm_gbs"], tf_burst=d["bf16_tflops"], tf_sust=d.get("bf16_tflops_sustained", d["bf16_tflops"]), src="measured")
    return dict(hbm=6650.0, tf_burst=1590.0, tf_sust=1400.0, src="fallback")   # B200_PROFILING.md fallback


def run_reference(args, cfg_index, cfg, rank, world):
    """--impl reference: the CPU oracle, as it stands, on a bounded sample of the workload (rank 0 only)."""
    if rank != 0:
        return
    from oracle import oracle
    arch = cfg["arch"]; T = min(cfg["T"], 2); B = min(cfg["B"], 2 if arch.kind == "impala" else 4)
    oa = oracle.make_arch(arch.kind, arch.channels, arch.fc, arch.n_actions, arch.in_c, arch.in_h, arch.in_w)
    kw = dict(epochs=1, minibatches=1) if cfg["algo"] == "ppo" else {}
    ho = oracle.make_hparams(cfg["algo"], T, B, lr=cfg["lr"], max_grad_norm=cfg["max_grad_norm"], **kw)
    sub = dict(cfg); sub["T"], sub["B"] = T, B
    bt = gen_inputs(cfg_index, sub, 1, 0)[0]
    params = synth.gen_params(arch, 1, head_scale=0.1); P = params.size
    m = np.zeros(P, np.float32); v = np.zeros(P, np.float32)
    times = []
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        oracle.learner_step(oa, ho, params, m, v, 0, bt["obs"], bt["actions"], bt["rewards"], bt["dones"], bt["behaviour_logits"])
        if i >= args.warmup:
            times.append(time.perf_counter() - t0)
    total = sum(times); value = T * B * len(times) / total
    sample = f"T={T}, B={B} envs of the workload per step ({(T + 1) * B} frames forward, {T * B} backward), full network, 1 thread"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * total / len(times), "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"BASELINE.json configs[{cfg_index}]", "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def cpu_baseline(cfg_index, cfg, budget_s=12.0):
    """The oracle as it stands, 1 thread, on a bounded sample of the same workload (about 10-30 s)."""
    from oracle import oracle
    arch = cfg["arch"]; T, B = 2, 2
    oa = oracle.make_arch(arch.kind, arch.channels, arch.fc, arch.n_actions, arch.in_c, arch.in_h, arch.in_w)
    kw = dict(epochs=1, minibatches=1) if cfg["algo"] == "ppo" else {}
    ho = oracle.make_hparams(cfg["algo"], T, B, lr=cfg["lr"], max_grad_norm=cfg["max_grad_norm"], **kw)
    sub = dict(cfg); sub["T"], sub["B"] = T, B
    bt = gen_inputs(cfg_index, sub, 1, 0)[0]
    params = synth.gen_params(arch, 1, head_scale=0.1); P = params.size
    n, t0 = 0, time.perf_counter()
    while True:
        oracle.learner_step(oa, ho, params, np.zeros(P, np.float32), np.zeros(P, np.float32), 0, bt["obs"], bt["actions"], bt["rewards"], bt["dones"], bt["behaviour_logits"])
        n += 1
        if time.perf_counter() - t0 > budget_s:
            break
    dt = time.perf_counter() - t0
    return {"value": T * B * n / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"{n} oracle learner steps at T={T}, B={B} ({(T + 1) * B} frames forward, {T * B} backward each), same network and loss, {dt:.1f} s"}


def read_traffic(cfg_index, cls):
    """dram bytes per launch of a kernel class from the committed `ncu --set full` summary (profiles/traffic.csv, written from the
    capture described in profiles/traffic.md); None if that class was not captured for this config."""
    tpath = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(tpath):
        for line in open(tpath).read().splitlines()[1:]:
            f = line.split(",")
            if len(f) == 3 and f[0] == str(cfg_index) and f[1] == cls:
                return float(f[2])
    return None


def roofline_of(dom, peaks, clk, t_local, cfg_index):
    bound = "tensor" if dom["flops"] > 0 else "hbm"
    per_launch_s = dom["ms"] / 1e3 / max(dom["launches"], 1)
    if bound == "tensor":
        achieved = dom["flops"] / dom["launches"] / per_launch_s / 1e12; runit = "TFLOP/s"
        peak, src = pick_tensor_peak(peaks, clk)
    else:
        achieved = dom["bytes"] / dom["launches"] / per_launch_s / 1e9; peak = peaks["hbm"]; runit = "GB/s"; src = f"{peaks['src']} (copy)"
    return {"bound": bound, "kernel": dom["name"], "achieved": achieved, "peak": peak, "unit": runit, "frac": achieved / peak,
            "traffic": read_traffic(cfg_index, dom["name"]), "traffic_source": "profiles/traffic.csv (ncu --set full capture, see profiles/traffic.md)",
            "peak_source": src, "launches": dom["launches"], "ms_per_launch": 1e3 * per_launch_s, "share_of_step": dom["ms"] / (1e3 * t_local)}


def measure_learner(cfg_index, cfg, steps, warmup, rank, local, world, use_dp, full):
    """Times `steps` learner steps of one BASELINE config.  full = the headline treatment (e2e with host buffers, inference);
    otherwise the short form used for `other_configs`."""
    import torch
    import torch.distributed as dist
    from paper_2310_00036_b200 import binding
    T, B, arch, prec = cfg["T"], cfg["B"], cfg["arch"], cfg["precision"]
    kw = {} if cfg["algo"] != "ppo" else dict(epochs=4, minibatches=4)
    hp = binding.make_hparams(cfg["algo"], prec, T, B, lr=cfg["lr"], max_grad_norm=cfg["max_grad_norm"], **kw)
    net = binding.Net(arch, max_frames=(T + 1) * B)
    learner = net
    if use_dp and world > 1:
        from paper_2310_00036_b200 import dp
        learner = dp.DataParallelLearner(net)
    params0 = synth.gen_params(arch, 1, head_scale=0.1)
    sets = gen_inputs(cfg_index, cfg, N_ROTATE, rank)
    keys = ("obs", "actions", "rewards", "dones", "behaviour_logits")
    host_sets = [{k: torch.from_numpy(s[k]).pin_memory() for k in keys} for s in sets]
    dev_sets = [{k: v.cuda(non_blocking=True) for k, v in hs.items()} for hs in host_sets]
    P = net.P
    dp_, dm, dv = torch.from_numpy(params0).cuda(), torch.zeros(P, device="cuda"), torch.zeros(P, device="cuda")
    n_upd = hp.epochs * hp.minibatches if hp.algo == 1 else 1
    stats = torch.zeros((n_upd, binding.N_STATS), device="cuda")
    stream = torch.cuda.current_stream()
    kstep = 0

    def step(i, bufs):
        nonlocal kstep
        s = bufs[i % len(bufs)]
        kstep, _ = learner.learner_step(dp_, dm, dv, kstep, s["obs"], s["actions"], s["rewards"], s["dones"], s["behaviour_logits"], hp, stats)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- warm-up; the second pass profiles every kernel class to find the dominant one ----------------------
    clocks = ClockSampler(local)      # started here: nvidia-smi takes longer to come up than a short timed region lasts
    step(0, dev_sets); torch.cuda.synchronize()
    binding.profile_begin(-1)
    step(1, dev_sets)
    prof_all = binding.profile_end()
    dominant = max(prof_all, key=lambda e: e["ms"])
    for i in range(2, warmup):
        step(i, dev_sets)
    # ---- timed region: K steps, inputs resident in HBM; events on the launching stream, one after every step ---
    barrier()
    l0 = binding.launch_count()
    binding.profile_begin(dominant["cls"])        # two events around each launch of the dominant class only
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    clocks.begin()
    ev[0].record(stream)
    for i in range(steps):
        step(i, dev_sets); ev[i + 1].record(stream)
    barrier()
    clocks.end()
    net.check_errors()
    t_local = ev[0].elapsed_time(ev[steps]) / 1e3
    per_step = [ev[i].elapsed_time(ev[i + 1]) for i in range(steps)]
    dom = binding.profile_end()[0]
    launches = binding.launch_count() - l0
    clk = clocks.stop()
    t = max_over_ranks(t_local, world)
    frames = sum_over_ranks(float(T * B * steps), world)
    loss_last = float(stats[-1, 0].item())
    assert np.isfinite(loss_last), "learner produced a non-finite loss"
    peaks = load_peaks()
    tpeak, _ = pick_tensor_peak(peaks, clk)
    flops = useful_flops_per_step(cfg)
    h2d = sum(v.numel() * v.element_size() for v in host_sets[0].values())
    res = {"value": frames / t, "ms_per_step": 1e3 * t / steps, "ms_per_step_median": statistics.median(per_step), "ms_per_step_min": min(per_step),
           "t_local": t_local, "launches": int(launches), "clocks": clk, "loss": loss_last, "h2d": int(h2d), "frames": frames,
           "tflops_useful": flops * steps / t_local / 1e12, "pct_bf16_tc_peak": 100.0 * flops * steps / t_local / 1e12 / tpeak,
           "roofline": roofline_of(dom, peaks, clk, t_local, cfg_index),
           "breakdown": {e["name"]: round(e["ms"], 4) for e in sorted(prof_all, key=lambda e: -e["ms"])}, "breakdown_total": sum(e["ms"] for e in prof_all)}
    if not full:
        net.close(); del dev_sets, host_sets
        torch.cuda.empty_cache()
        return res

    # ---- end to end through the public API with HOST buffers: H2D of the step's inputs + D2H of its stats ---
    d2h = stats.numel() * 4
    stats_host = torch.empty(stats.shape, dtype=torch.float32).pin_memory()
    # two device staging sets and a copy stream: the pinned-host -> device copy of step i+1 is issued before step i is launched, the
    # way a training loop prefetches its next batch; every step's inputs still cross the bus and every step's loss is read back
    # inside the timed region
    stages = [{k: torch.empty_like(v, device="cuda") for k, v in host_sets[0].items()} for _ in range(2)]
    ready = [torch.cuda.Event(), torch.cuda.Event()]
    copy_stream = torch.cuda.Stream()
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)

    def issue_copy(i):
        hs, st = host_sets[i % len(host_sets)], stages[i % 2]
        with torch.cuda.stream(copy_stream):
            for k in keys:
                st[k].copy_(hs[k], non_blocking=True)
            ready[i % 2].record(copy_stream)

    def e2e_step(i, last):
        nonlocal kstep
        if not last:
            issue_copy(i + 1)          # buffer (i+1) % 2 was last read by step i-1, which has completed (synchronised below)
        st = stages[i % 2]
        stream.wait_event(ready[i % 2])
        kstep, _ = learner.learner_step(dp_, dm, dv, kstep, st["obs"], st["actions"], st["rewards"], st["dones"], st["behaviour_logits"], hp, stats)
        stats_host.copy_(stats, non_blocking=True)
        stream.synchronize()        # the caller reads the loss every step
        return float(stats_host[-1, 0])

    issue_copy(0); e2e_step(0, True)
    barrier()
    w0 = time.perf_counter(); e0.record(stream)
    issue_copy(0)
    for i in range(steps):
        e2e_step(i, i + 1 == steps)
    e1.record(stream)
    barrier()
    t_e2e = max_over_ranks(max(e0.elapsed_time(e1) / 1e3, time.perf_counter() - w0), world)
    res["e2e"] = {"value": frames / t_e2e, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h)}

    # ---- actor side (BASELINE.json configs[1]): policy/value inference + Gumbel-max sampling, B = 128, bf16 mode ----
    if rank == 0 and arch.kind == "impala":
        Bi = 128
        anet = binding.Net(arch, max_frames=Bi)      # an actor owns its own net (cleanba.h: a cb_net is single-role)
        obs_i = [dev_sets[i % len(dev_sets)]["obs"].reshape(-1, arch.in_c, arch.in_h, arch.in_w)[j * Bi:(j + 1) * Bi].contiguous()
                 for i in range(N_ROTATE) for j in range(4)]
        for i in range(3 * len(obs_i)):      # steady state of a rollout loop: every observation buffer has been seen (third call on: graph replay)
            anet.policy_forward(dp_ if i == 0 else None, obs_i[i % len(obs_i)], seed=1, step=i, precision=prec)
        torch.cuda.synchronize()
        li = binding.launch_count(); ncall = 100
        e0.record(stream)
        for i in range(ncall):      # a rollout of T steps uses one parameter version (Figure 1): weights are packed on its first step only
            anet.policy_forward(dp_ if i % T == 0 else None, obs_i[i % len(obs_i)], seed=1, step=i, precision=prec)
        e1.record(stream); torch.cuda.synchronize()
        anet.check_errors()
        us = 1e3 * e0.elapsed_time(e1) / ncall
        res["inference"] = {"workload": f"BASELINE.json configs[1]: IMPALA-ResNet policy/value forward + Gumbel-max sampling, B=128, bf16 mode, new parameters every {T} calls",
                            "us_per_call": us, "env_frames_per_s": Bi / (us * 1e-6), "launches_per_call": (binding.launch_count() - li) / ncall}
        anet.close()
    net.close(); del dev_sets, host_sets, stages
    torch.cuda.empty_cache()
    return res


def measure_hbm_kernels(peaks):
    """The HBM-bound kernels of the path (scans, losses, norm, optimizer) through their own C-ABI entry points, at the
    BASELINE shapes (launch-latency bound by construction: <= 0.7 MB) and at a scaled-up shape whose working set exceeds the L2
    (T = 128, B = 65 536 trajectories; P = 64 M parameters), so that the kernels themselves are characterised.  Times come from the
    library's per-class CUDA events (two events around every launch).  bytes = algorithmic bytes (operands read once + results written once)."""
    import torch
    from paper_2310_00036_b200 import binding
    out = []
    A = 18
    g = torch.Generator(device="cuda"); g.manual_seed(5)

    def run(name, shape, fn, reps, classes):
        fn(); fn(); torch.cuda.synchronize()
        binding.profile_begin(-1)
        for _ in range(reps):
            fn()
        prof = {e["name"]: e for e in binding.profile_end()}
        for c in classes:
            e = prof[c]; us = 1e3 * e["ms"] / e["launches"]; by = e["bytes"] / e["launches"]
            out.append({"kernel": name if len(classes) == 1 else f"{name}:{c}", "class": c, "shape": shape, "bytes": by, "us": us, "GBps": by / us / 1e3,
                        "frac_hbm": by / us / 1e3 / peaks["hbm"], "launches_per_call": e["launches"] / reps})

    for label, T, B, P, reps in (("BASELINE shape", 20, 128, 1094115, 20), ("scaled-up shape", 128, 65536, 64 * 1024 * 1024, 5)):
        N = T * B
        V = torch.randn((T + 1, B), device="cuda", generator=g); r = torch.randn((T, B), device="cuda", generator=g)
        d = (torch.rand((T, B), device="cuda", generator=g) < 0.02).to(torch.uint8)
        lpi = -torch.rand((T, B), device="cuda", generator=g) - 1; lmu = lpi + 0.3 * torch.randn((T, B), device="cuda", generator=g)
        shp = f"{label}: T={T}, B={B}"
        run("vtrace", shp, lambda: binding.vtrace(V, r, d, lpi, lmu), reps, ["scan"])
        run("gae", shp, lambda: binding.gae(V, r, d), reps, ["scan"])
        head = torch.randn((N, A + 1), device="cuda", generator=g); act = torch.randint(0, A, (N,), device="cuda", generator=g, dtype=torch.int32)
        head_l = head[:, :A].contiguous()
        run("logprob_entropy", f"{label}: N={N}, A={A}", lambda: binding.logprob_entropy(head_l, act), reps, ["logprob"])
        vs = torch.randn(N, device="cuda", generator=g); pg = torch.randn(N, device="cuda", generator=g); rho = torch.rand(N, device="cuda", generator=g)
        buf = binding._loss_out(head, "bf16")
        run("impala_loss", f"{label}: N={N}, A={A}, bf16 seeds", lambda: binding.impala_loss(head, act, vs, pg, rho, precision="bf16", out=buf), reps, ["loss", "stats"])
        lpo = -torch.rand(N, device="cuda", generator=g) - 1
        run("ppo_loss", f"{label}: m={N}, A={A}, bf16 seeds", lambda: binding.ppo_loss(head, None, act, vs, pg, lpo, precision="bf16", out=buf), reps, ["loss"])
        del head, head_l, buf, vs, pg, rho, lpo, V, r, d, lpi, lmu
        th = torch.randn(P, device="cuda", generator=g) * 0.05; m = torch.zeros(P, device="cuda"); v = torch.zeros(P, device="cuda")
        gr = torch.randn(P, device="cuda", generator=g) * 1e-3
        scratch = torch.empty(P // 4096 + 16, dtype=torch.float64, device="cuda")
        k = [0]

        def adam():
            k[0] += 1
            binding.clip_adam(th, m, v, gr, k[0], 6e-4, scratch=scratch)
        run("clip_adam", f"{label}: P={P}", adam, reps, ["sqnorm", "adam"])
        del th, m, v, gr, scratch
        torch.cuda.empty_cache()
    return out


def measure_pipeline(cfg, iters=10):
    """Cleanba's actor/learner architecture (cb_pipeline: Figure 1 right / Table 1) against the Synchronous architecture on the config's
    shapes: device time per iteration (one rollout of T steps on B envs with the on-device synthetic environment + one learner call)."""
    import torch
    from paper_2310_00036_b200 import binding
    T, B, arch, prec = cfg["T"], cfg["B"], cfg["arch"], cfg["precision"]
    kw = {} if cfg["algo"] != "ppo" else dict(epochs=4, minibatches=4)
    hp = binding.make_hparams(cfg["algo"], prec, T, B, lr=cfg["lr"], max_grad_norm=cfg["max_grad_norm"], **kw)
    params = torch.from_numpy(synth.gen_params(arch, 1, head_scale=0.1)).cuda()
    res = {}
    for name, sync in (("synchronous", True), ("cleanba", False)):
        pipe = binding.Pipeline(arch, hp, params, sync=sync, env_seed=11, sample_seed=12)
        pipe.run(4); pipe.wait()
        pipe.run(iters); ms = pipe.wait()
        rec = pipe.records(3)
        res[name] = {"ms_per_iteration": ms / iters, "env_frames_per_s": T * B / (ms / iters * 1e-3), "last_record": list(rec[-1])}
        pipe.close()
    res["overlap_gain"] = 1.0 - res["cleanba"]["ms_per_iteration"] / res["synchronous"]["ms_per_iteration"]
    res["workload"] = f"{iters} iterations of rollout (T={T} policy steps on B={B} on-device synthetic envs) + learner call, {cfg['algo']}, {prec} mode; last_record = (iteration, data policy version, learner version before, after)"
    torch.cuda.empty_cache()
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config index (2, 3, 4; 0 = small parity case)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--dp", action="store_true", help="N > 1: one data-parallel learner over all ranks instead of N replicas")
    ap.add_argument("--only", default="", help="comma list out of: learner, other, hbm, pipeline (default: everything); for profiler runs")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0")); local = int(os.environ.get("LOCAL_RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    cfg = workload(args.config)
    if args.impl == "reference":
        return run_reference(args, args.config, cfg, rank, world)

    import torch
    from paper_2310_00036_b200 import binding, build
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    binding.lib()
    only = set(x for x in args.only.split(",") if x) or {"learner", "other", "hbm", "pipeline"}
    warmup = max(args.warmup, 3); steps = max(args.steps, 1)
    T, B, arch, prec = cfg["T"], cfg["B"], cfg["arch"], cfg["precision"]
    peaks = load_peaks()
    line = {"metric": METRIC, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "bf16" if prec == "bf16" else "f32", "data": "synthetic"}
    if "learner" in only:
        r = measure_learner(args.config, cfg, steps, warmup, rank, local, world, args.dp, True)
        par = "1 gpu" if world == 1 else (f"dp{world}: {B} envs per rank, one fixed-order gradient exchange per update" if args.dp else "replicas only")
        line.update({
            "value": r["value"], "ms_per_step": r["ms_per_step"], "ms_per_step_median": r["ms_per_step_median"], "ms_per_step_min": r["ms_per_step_min"],
            "config": {"workload": f"BASELINE.json configs[{args.config}]: {cfg['algo']} learner step, {net_key(arch)} net, T={T}, B={B}, {prec} mode",
                       "frames_per_step": T * B, "parallelism": par,
                       "l2": f"{N_ROTATE} input sets of {r['h2d'] / 1e6:.0f} MB rotated (> 126 MB L2 together with the activations)"},
            "tflops_useful": r["tflops_useful"], "pct_bf16_tc_peak": r["pct_bf16_tc_peak"], "clocks": r["clocks"], "gpu_launches": r["launches"],
            "e2e": r["e2e"], "roofline": r["roofline"], "kernel_breakdown_ms_per_step": r["breakdown"], "kernel_breakdown_total_ms": r["breakdown_total"],
            "loss": r["loss"], "inference": r.get("inference")})
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    if world == 1:
        if "other" in only:      # the PPO iteration and the wide network, a few steps each (the headline stays the metric's config)
            oc = {}
            for ci in (3, 4):
                if ci == args.config:
                    continue
                c = synth.CONFIGS[ci]
                r = measure_learner(ci, c, 5, 3, 0, local, 1, False, False)
                oc[str(ci)] = {"workload": f"BASELINE.json configs[{ci}]: {c['algo']} learner {'iteration (16 updates)' if c['algo'] == 'ppo' else 'step'}, {net_key(c['arch'])} net, T={c['T']}, B={c['B']}, {c['precision']} mode",
                               "steps": 5, "warmup": 3, "ms_per_step": r["ms_per_step"], "ms_per_step_min": r["ms_per_step_min"], "value": r["value"], "unit": UNIT,
                               "tflops_useful": r["tflops_useful"], "pct_bf16_tc_peak": r["pct_bf16_tc_peak"], "clocks": r["clocks"], "gpu_launches": r["launches"],
                               "roofline": r["roofline"], "kernel_breakdown_ms_per_step": r["breakdown"]}
            line["other_configs"] = oc
        if "hbm" in only:
            line["hbm_kernels"] = measure_hbm_kernels(peaks)
        if "pipeline" in only and arch.kind == "impala":
            line["pipeline"] = measure_pipeline(cfg)
    if not args.no_cpu_baseline and "learner" in only:
        line["cpu_baseline"] = cpu_baseline(args.config, cfg)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
