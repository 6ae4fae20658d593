"""Host logic of the sharded path (paper_2105_08026_b200/sharded.py) on CPU: the driver and
its exchange are exercised with the ORACLE as the engine (same two calls as the CUDA binding: shard_sweep /
shard_decide), in one process and across two gloo ranks.  A sharded chain must be the unsharded chain: same Philox
streams (keyed by the global object index), same theta decisions (sums differ only in their order)."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

from oracle import api as O
from paper_2105_08026_b200 import sharded, synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shard_ranges_are_even_and_cover():
    for n, g in ((1000, 2), (1001, 3), (7, 4), (300_000, 8), (5, 8)):
        rs = sharded.shard_ranges(n, g)
        assert rs[0][0] == 0 and rs[-1][1] == n and all(a[1] == b[0] for a, b in zip(rs, rs[1:]))
        assert all(lo % 2 == 0 for lo, hi in rs if hi > lo)


def _engines(model, inp, n, ranges, seed, astar, **kw):
    out = []
    for lo, hi in ranges:
        e = O.Sampler(model, hi - lo, seed=seed, target_accept_chi=astar, object_offset=lo, n_objects_total=n, **kw)
        e.set_data([c[lo:hi] for c in inp["cols"]])
        if inp["consts"] is not None:
            e.set_model_consts(inp["consts"])
        e.set_init(inp["theta0"])
        out.append(e)
    return out


@pytest.mark.parametrize("model,maker,astar,n", [(0, synth.make_normal1d, 0.44, 401), (1, synth.make_thinned_schechter1d, 0.44, 300),
                                                  (4, synth.make_bb1_fluxnoise1d, 0.44, 250), (5, synth.make_normal3d_knowncov, 0.234, 333)],
                         ids=["M0", "M1", "M4", "M5"])
def test_three_local_shards_reproduce_the_unsharded_chain(model, maker, astar, n):
    inp = maker(n, 80 + model)
    iters, burn, thin = 150, 30, 4
    whole = _engines(model, inp, n, [(0, n)], 80 + model, astar, keep_chi_moments=True)[0]
    whole.run(iters, burn, thin)
    parts = _engines(model, inp, n, sharded.shard_ranges(n, 3), 80 + model, astar, keep_chi_moments=True)
    sharded.LocalShards(parts).run(iters, burn, thin)
    for e in parts:                                            # theta is replicated: identical on every shard
        np.testing.assert_allclose(e.get_theta_trace(), whole.get_theta_trace(), rtol=1e-9, atol=1e-10)
        assert np.array_equal(e.get_theta_trace(), parts[0].get_theta_trace())
    chi = np.concatenate([e.get_state()["chi"] for e in parts], axis=1)
    L = np.concatenate([e.get_state()["L"] for e in parts], axis=1)
    np.testing.assert_allclose(chi, whole.get_state()["chi"], rtol=1e-9, atol=1e-10)
    np.testing.assert_allclose(L, whole.get_state()["L"], rtol=1e-9)
    mean = np.concatenate([e.get_chi_moments()[0] for e in parts], axis=1)
    np.testing.assert_allclose(mean, whole.get_chi_moments()[0], rtol=1e-9, atol=1e-10)
    sw, sp = whole.get_stats(), parts[0].get_stats()
    assert sp["chi_accepts"] == sw["chi_accepts"] and sp["theta_accepts"] == sw["theta_accepts"]
    assert sp["chi_proposals"] == sw["chi_proposals"] == iters * n


WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import numpy as np
import torch.distributed as dist
from oracle import api as O
from paper_2105_08026_b200 import sharded, synth
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
n = 300
inp = synth.make_thinned_schechter1d(n, 91)
lo, hi = sharded.shard_ranges(n, world)[rank]
e = O.Sampler(1, hi - lo, seed=91, target_accept_chi=0.44, object_offset=lo, n_objects_total=n)
e.set_data([c[lo:hi] for c in inp["cols"]]); e.set_model_consts(inp["consts"]); e.set_init(inp["theta0"])
sharded.DistributedShard(e, dist).run(120, 20, 5)
dist.barrier()
print(json.dumps(dict(rank=rank, trace=e.get_theta_trace().tolist(), chi=e.get_state()["chi"][0].tolist(),
                      acc=e.get_stats()["chi_accepts"])))
dist.destroy_process_group()
"""


def test_two_gloo_ranks_reproduce_the_unsharded_chain(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29631", WORLD_SIZE="2")
    procs = [subprocess.Popen([sys.executable, str(script)], env=dict(env, RANK=str(r)), stdout=subprocess.PIPE,
                              stderr=subprocess.PIPE, text=True) for r in range(2)]
    outs = [p.communicate(timeout=300) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    res = sorted((json.loads(o[0].strip().splitlines()[-1]) for o in outs), key=lambda d: d["rank"])
    n = 300
    inp = synth.make_thinned_schechter1d(n, 91)
    whole = O.Sampler(1, n, seed=91, target_accept_chi=0.44)
    whole.set_data(inp["cols"]); whole.set_model_consts(inp["consts"]); whole.set_init(inp["theta0"])
    whole.run(120, 20, 5)
    assert res[0]["trace"] == res[1]["trace"]                  # both ranks took identical decisions, bit for bit
    np.testing.assert_allclose(np.array(res[0]["trace"]), whole.get_theta_trace(), rtol=1e-9, atol=1e-10)
    np.testing.assert_allclose(np.concatenate([res[0]["chi"], res[1]["chi"]]), whole.get_state()["chi"][0], rtol=1e-9, atol=1e-10)
    assert res[0]["acc"] == res[1]["acc"] == whole.get_stats()["chi_accepts"]
