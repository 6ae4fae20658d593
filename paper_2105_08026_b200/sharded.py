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

from . import binding

# layout of the totals vector: {S, Delta, Tq, n_accept, n_nonfinite}; Tq (the selection sum of M1 / M4) is computed in
# full by every shard and is NOT summed -- the rule lives in the library (cudahm_shard_combine)


def shard_ranges(n_total, n_shards):
    """Contiguous object ranges [lo, hi) with EVEN boundaries (objects draw their random numbers in pairs)."""
    per = -(-n_total // n_shards)
    per += per & 1
    return [(min(r * per, n_total), min((r + 1) * per, n_total)) for r in range(n_shards)]


def combine(totals_by_rank):
    """Fixed-order (rank-order) sum of the per-shard totals: cudahm_shard_combine (host code of the library)."""
    return binding.shard_combine(np.asarray(totals_by_rank, dtype=np.float64))


class LocalShards:
    """Several shards driven from one process (e.g. two handles on one GPU, launched one after the other).  With
    device=True (CUDA engines) the totals never visit the host between the sweep and the decision: every engine leaves its
    five totals in one device array, which each engine's shard_decide_gathered reads back once."""

    def __init__(self, engines, device=False):
        self.engines = list(engines)
        self.device = bool(device)
        if self.device:
            import torch
            self._gathered = torch.zeros((len(self.engines), 5), dtype=torch.float64, device=self.engines[0].device)

    def run(self, n_iter, burn_in=0, thin=1):
        for _ in range(int(n_iter)):
            if self.device:
                for r, e in enumerate(self.engines):
                    e.shard_sweep_device(self._gathered[r].data_ptr(), burn_in, thin)
                for e in self.engines:
                    e.shard_decide_gathered(self._gathered.data_ptr(), len(self.engines), burn_in, thin)
            else:
                tot = combine([e.shard_sweep(burn_in, thin) for e in self.engines])
                for e in self.engines:
                    e.shard_decide(tot, burn_in, thin)


class DistributedShard:
    """One shard per process; `dist` is an initialised torch.distributed module.  Backend nccl with a CUDA engine: the
    shard's totals stay on the device, ONE all-gather on the sampler's stream, ONE read-back of 40 x world bytes inside
    cudahm_shard_decide_gathered.  Backend gloo (the CPU tests, oracle engines): host buffers."""

    def __init__(self, engine, dist, device="cpu"):
        import torch
        self.engine, self.dist, self.torch, self.device = engine, dist, torch, device
        self.world = dist.get_world_size()
        self.on_device = str(device).startswith("cuda") and hasattr(engine, "shard_sweep_device")
        if self.on_device:
            self._mine = torch.zeros(5, dtype=torch.float64, device=device)
            self._all = torch.zeros((self.world, 5), dtype=torch.float64, device=device)
        else:
            self._buf = [torch.empty(5, dtype=torch.float64) for _ in range(self.world)]

    def run(self, n_iter, burn_in=0, thin=1):
        torch = self.torch
        for _ in range(int(n_iter)):
            if self.on_device:
                self.engine.shard_sweep_device(self._mine.data_ptr(), burn_in, thin)
                self.dist.all_gather_into_tensor(self._all, self._mine)
                self.engine.shard_decide_gathered(self._all.data_ptr(), self.world, burn_in, thin)
            else:
                mine = torch.from_numpy(np.asarray(self.engine.shard_sweep(burn_in, thin), dtype=np.float64))
                self.dist.all_gather(self._buf, mine)
                self.engine.shard_decide(combine([b.numpy() for b in self._buf]), burn_in, thin)
