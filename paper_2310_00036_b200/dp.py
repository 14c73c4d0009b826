"""Data-parallel learner ("multiple learner devices via pmap", 350-366: App. A Option 2, every
device runs Algorithm 1 on its own environments and the gradients of the copies are averaged before the optimizer step).

One process per GPU (torch.distributed).  Per gradient update: cb_learner_grad on the local envs, ONE exchange of the flat fp32
gradient, cb_learner_apply -- so every rank applies the same bytes and the replicas stay bit-identical.  The exchange is a
reduce-scatter + all-gather written so that the floating-point association is fixed: an all-to-all hands rank r chunk r of every
rank's gradient, ordered by source rank; cb_sum_ranks adds the G chunks in rank order (the library's kernel) and scales by 1/G; an
all-gather returns the averaged chunks.  Nothing here depends on the collective library's own reduction order.
Marshalling only: every arithmetic step runs in the library's kernels.
"""
import torch
import torch.distributed as dist


def chunk_elems(P, world):
    """Elements per rank chunk: ceil(P / world) rounded up to a multiple of 4 (16-byte vector loads in cb_sum_ranks)."""
    n = (P + world - 1) // world
    return (n + 3) // 4 * 4


class GradientExchange:
    """Averages a flat fp32 gradient over the ranks of `group`, in place, bitwise identically on every rank."""

    def __init__(self, P, device, group=None, sum_fn=None):
        self.P, self.group = P, group
        self.world = dist.get_world_size(group); self.rank = dist.get_rank(group)
        self.n = chunk_elems(P, self.world)
        self.send = torch.zeros(self.world * self.n, dtype=torch.float32, device=device)
        self.recv = torch.empty((self.world, self.n), dtype=torch.float32, device=device)
        self.red = torch.empty(self.n, dtype=torch.float32, device=device)
        self.full = torch.empty(self.world * self.n, dtype=torch.float32, device=device)
        if sum_fn is None:
            from . import binding
            sum_fn = binding.sum_ranks               # cb_sum_ranks: the only arithmetic of the exchange
        self.sum_fn = sum_fn

    def __call__(self, grad):
        self.send[:self.P].copy_(grad)              # the tail beyond P stays zero
        dist.all_to_all_single(self.recv.view(-1), self.send, group=self.group)      # row s of recv = chunk `rank` of rank s's gradient
        self.sum_fn(self.recv, 1.0 / self.world, out=self.red)
        dist.all_gather_into_tensor(self.full, self.red, group=self.group)
        grad.copy_(self.full[:self.P])
        return grad


class DataParallelLearner:
    """cb_learner_step over the envs of ALL ranks: each rank passes its own B_local envs; returns like Net.learner_step."""

    def __init__(self, net, group=None):
        self.net = net
        self.exchange = GradientExchange(net.P, "cuda", group)

    def learner_step(self, params, adam_m, adam_v, opt_step, obs, actions, rewards, dones, behaviour_logits, hp, stats=None, behaviour_values=None):
        n, stats, h = self.net.learner_begin(params, adam_m, adam_v, opt_step, obs, actions, rewards, dones, behaviour_logits, hp, stats, behaviour_values)
        for u in range(n):
            g = self.net.learner_grad(u)
            self.exchange(g)
            self.net.learner_apply(u)
        return h.opt_step, stats
