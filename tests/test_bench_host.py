"""Host logic of bench.py: the replicas-only aggregation over ranks (world_size 2, gloo, CPU) and the helpers."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
rank = int(os.environ["RANK"])
dist.init_process_group("gloo", rank=rank, world_size=int(os.environ["WORLD_SIZE"]))
# rank 0: 1000 units in 2 ms; rank 1: 3000 units in 4 ms  ->  4000 units / 4 ms (max over ranks)
value, ms, units = bench.aggregate([2.0, 4.0][rank], [1000.0, 3000.0][rank], dist)
dist.barrier()
if rank == 0:
    print(json.dumps(dict(value=value, ms=ms, units=units)))
dist.destroy_process_group()
"""


def test_aggregate_world_size_2_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29617", WORLD_SIZE="2")
    procs = [subprocess.Popen([sys.executable, str(script)], env=dict(env, RANK=str(r)), stdout=subprocess.PIPE,
                              stderr=subprocess.PIPE, text=True) for r in range(2)]
    outs = [p.communicate(timeout=240) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    res = json.loads(outs[0][0].strip().splitlines()[-1])
    assert res["ms"] == 4.0 and res["units"] == 4000.0
    assert res["value"] == pytest.approx(4000.0 / 4e-3)


def test_aggregate_single_process():
    sys.path.insert(0, ROOT)
    import bench
    v, ms, u = bench.aggregate(2.0, 1000.0, None)
    assert (v, ms, u) == (1000.0 / 2e-3, 2.0, 1000.0)
    assert bench.trace_rows_needed(10000, 2000, 10) == 801
    c, n, inp = bench.make_workload("C0")
    assert n == 1000 and len(inp["cols"]) == 2
    r = bench.roofline_entry("C2", bench.synth.CONFIGS["C2"], 300000, 100, 0, 1.0, 6547.5, "x")
    assert r["alg_bytes_per_iter"] == 24_000_000 and r["frac"] == pytest.approx(24e6 * 100 / 1e-3 / 1e9 / 6547.5)
