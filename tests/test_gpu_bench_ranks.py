"""-m gpu: bench.py under torchrun with two ranks. The box has one GPU, so both ranks run on GPU 0 and the collectives
(barrier, max / sum of the timings) go through gloo (MKF_BENCH_BACKEND / MKF_BENCH_ONE_GPU of bench.py): the ranks own
independent workloads and no kernel of one waits for the other, so this tests the plumbing every rank goes through
(same number of barriers on every rank, one JSON line from rank 0, units summed), not a throughput."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(extra, port):
    env = dict(os.environ, MKF_BENCH_BACKEND="gloo", MKF_BENCH_ONE_GPU="1", MKF_BENCH_SERIAL="1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), "bench.py", "--gpus", "2", "--steps", "2", "--warmup", "3", "--no-cpu-baseline",
           "--e2e-steps", "1"] + extra
    r = subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-3000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                     # rank 0 alone prints
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["scaling"] == "weak" and d["value"] > 0 and d["gpu_launches"] > 0
    return d


def test_bench_headline_with_two_ranks():
    d = _run(["--scale", "0.02"], 29533)                       # the default line at N > 1: the fit on configs[1]
    one = 4000000 * 0.02 * 17                                  # layer-steps of one rank's workload, at most
    assert one < d["units_per_step"] <= 2 * one               # both ranks' units are in the sum
    assert d["e2e"]["value"] > 0 and d["roofline"]["bound"] == "alu"


def test_bench_build_with_two_ranks_and_rank0_only_extras():
    d = _run(["--workload", "build3", "--scale", "0.05"], 29534)
    assert d["units_per_step"] == 20.0                        # 10 events per rank
    assert d["chained_fit"]["value"] > 0 and d["overlap_recovery"]["value"] > 0     # measured by rank 0 alone, without barriers
