"""The N > 1 path of bench.py on CPU (gloo, world_size 2): the path has no data-path exchange
(replicas only), so what there is to test is the plumbing -- rank
environment, max-over-ranks timing, whole-job sums -- and that the reference arm runs on rank 0
alone under torchrun."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
rank, local_rank, world = bench.dist_env()
dist.init_process_group("gloo")
assert world == 2 and dist.get_world_size() == 2 and rank == dist.get_rank()
# timing is the MAX over ranks, throughput units are the SUM (whole-job aggregate)
t = bench.max_over_ranks(10.0 + 5.0 * rank, world)
u = bench.sum_over_ranks(100.0 * (rank + 1), world)
assert t == 15.0 and u == 300.0, (t, u)
# identity without a process group
assert bench.max_over_ranks(3.5, 1) == 3.5 and bench.sum_over_ranks(3.5, 1) == 3.5
dist.barrier()
if rank == 0:
    print(json.dumps(dict(ok=True, t=t, u=u)))
dist.destroy_process_group()
"""


def _torchrun(args, timeout=600):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="2")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29617"] + args
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def test_rank_aggregation_gloo_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    r = _torchrun([str(script)])
    assert r.returncode == 0, r.stderr[-2000:]
    line = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(line) == 1 and json.loads(line[0]) == dict(ok=True, t=15.0, u=300.0)


def test_reference_arm_under_torchrun_runs_on_rank0_only():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--workload", "C0"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                   # rank 1 exits 0 without work or output
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0 and d["unit"] == "interactions/s"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["config"]["workload"].startswith("C0")
