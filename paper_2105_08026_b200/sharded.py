"""Sharded populations over several samplers (one per GPU): SURVEY.md 8(e) / 8(f) NEXT-3, the paper's outlook of ~1e8
objects on a modest GPU cluster.

Objects are conditionally independent given theta (Eq. 2.4), so the plate shards by object range with no
data movement; theta, L_theta and the theta Philox stream are replicated, every rank takes the identical theta decision,
and the only exchange per Gibbs iteration is the sum of five doubles per rank.  The exchange is an all-gather followed
by a sum in RANK ORDER on every rank (deterministic, and the same bits everywhere), through `torch.distributed` (NCCL
between GPUs, gloo in the CPU tests) or, for several shards inside one process, a plain loop.  Argument marshalling
and the exchange only: every step of the path runs in the engines' kernels (`cudahm_shard_sweep / cudahm_shard_decide`).
"""
import numpy as np

# indices of the totals vector {S, Delta, Tq, n_accept, n_nonfinite}; Tq (the selection sum of M1 / M4) is computed in
# full by every shard and is NOT summed
SUMMED = (0, 1, 3, 4)


def shard_ranges(n_total, n_shards):
    """Contiguous object ranges [lo, hi) with EVEN boundaries (objects draw their random numbers in pairs)."""
    per = -(-n_total // n_shards)
    per += per & 1
    return [(min(r * per, n_total), min((r + 1) * per, n_total)) for r in range(n_shards)]


def combine(totals_by_rank):
    """Fixed-order (rank-order) sum of the per-shard totals; Tq taken from the first shard."""
    out = np.array(totals_by_rank[0], dtype=np.float64, copy=True)
    for t in totals_by_rank[1:]:
        for q in SUMMED:
            out[q] += t[q]
    return out


class LocalShards:
    """Several shards driven from one process (e.g. two handles on one GPU, launched one after the other)."""

    def __init__(self, engines):
        self.engines = list(engines)

    def run(self, n_iter, burn_in=0, thin=1):
        for _ in range(int(n_iter)):
            tot = combine([e.shard_sweep(burn_in, thin) for e in self.engines])
            for e in self.engines:
                e.shard_decide(tot, burn_in, thin)


class DistributedShard:
    """One shard per process; `dist` is an initialised torch.distributed module (backend nccl or gloo)."""

    def __init__(self, engine, dist, device="cpu"):
        import torch
        self.engine, self.dist, self.torch, self.device = engine, dist, torch, device
        self.world = dist.get_world_size()
        self._buf = [torch.empty(5, dtype=torch.float64, device=device) for _ in range(self.world)]

    def run(self, n_iter, burn_in=0, thin=1):
        torch = self.torch
        for _ in range(int(n_iter)):
            mine = torch.from_numpy(self.engine.shard_sweep(burn_in, thin)).to(self.device)
            self.dist.all_gather(self._buf, mine)
            tot = combine([b.cpu().numpy() for b in self._buf])
            self.engine.shard_decide(tot, burn_in, thin)
