"""N > 1 plumbing of bench.py on CPU: two gloo ranks own disjoint workloads (no data-path collective) and only
the timings / unit counts are reduced (max / sum)."""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import numpy as np, torch, torch.distributed as dist
import bench
from workloads import datagen
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
seed = bench.rank_seed(7, rank)
geom, prm, hits, seeds, _ = bench.make_fit_workload(seed, 0.0005)           # 2000 helices per rank
units = float((seeds["track_hits"] >= 0).sum())
ms, tot = bench.aggregate(10.0 + rank, units, world, "cpu")
first = float(seeds["par"][3, 0])
allfirst = [None] * world
dist.all_gather_object(allfirst, (first, units))
if rank == 0:
    print(json.dumps(dict(ms=ms, tot=tot, firsts=allfirst)))
dist.destroy_process_group()
"""


def test_two_gloo_ranks_shard_without_data_exchange(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29571", WORLD_SIZE="2")
    procs = [subprocess.Popen([sys.executable, str(script)], env=dict(env, RANK=str(r), LOCAL_RANK=str(r)),
                              stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True) for r in range(2)]
    outs = [p.communicate(timeout=300) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    import json
    d = json.loads(outs[0][0].strip().splitlines()[-1])
    assert d["ms"] == 11.0                                        # max over ranks
    (f0, u0), (f1, u1) = d["firsts"]
    assert d["tot"] == u0 + u1                                    # sum over ranks
    assert f0 != f1                                               # the ranks own different workloads


def test_aggregate_is_identity_for_one_rank():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate(3.5, 100.0, 1, "cpu") == (3.5, 100.0)
    assert bench.rank_seed(5, 3) == 8
