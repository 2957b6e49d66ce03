"""The N > 1 path on CPU (gloo, world_size 2): bench.py's rank plumbing (rank environment, max-over-ranks timing,
whole-job sums, the reference arm on rank 0 alone under torchrun) and the target sharding of the matvec
(DESIGN.md section 9): the library's partition rule (host-only C call) and the all-gather of the owned rows of y --
the one exchange step per matvec -- through the layout of paper_1810_03698_b200/shard.py, which the GPU tests tie to
the kernels."""
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


def test_shard_partition_rule():
    """pb_shard_partition (host-only): boundaries are monotone, cover every group, are the same on every rank (a pure
    function of the costs) and cut the prefix sum within one group's cost of k/world of the total."""
    import numpy as np
    from paper_1810_03698_b200 import pb
    pb.build()
    rng = np.random.Generator(np.random.PCG64(5))
    for G, world in ((1, 1), (7, 2), (100, 3), (16211, 8), (5, 8), (64, 64)):
        cost = rng.integers(0, 10_000, size=G)
        first = pb.shard_partition(cost, world)
        assert first[0] == 0 and first[-1] == G and np.all(np.diff(first) >= 0)
        pre = np.concatenate([[0], np.cumsum(cost)])
        for k in range(1, world):
            want = pre[-1] * k / world
            assert pre[first[k]] >= want - 1e-9 and (first[k] == 0 or pre[first[k] - 1] < want + 1e-9)
        if G >= 8 * world:
            share = np.diff(pre[first])
            assert share.max() <= pre[-1] / world + cost.max()
    assert np.array_equal(pb.shard_partition(np.zeros(10, dtype=np.int64), 4), [0, 0, 0, 0, 10])   # nothing to balance
    with pytest.raises(pb.PBError):
        pb.shard_partition(np.array([3, -1, 2]), 2)


_SHARD_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import numpy as np, torch, torch.distributed as dist
from paper_1810_03698_b200 import pb, shard
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
# every rank derives the SAME partition from the same per-group costs (no communication)
N, TG = 1000, 64                                        # ragged: 15 full groups + one of 40 panels
G = (N + TG - 1) // TG
cost = np.random.Generator(np.random.PCG64(11)).integers(1, 1000, size=G)
first = shard.group_ranges_to_panels(pb.shard_partition(cost, world), N, TG)
perm = np.random.Generator(np.random.PCG64(12)).permutation(N)            # Morton position -> original panel
y_morton = np.random.Generator(np.random.PCG64(13)).normal(size=(2, N))    # stands for the rows each rank would compute
mine = y_morton.copy()
mine[:, :first[rank]] = np.nan                                             # a rank only has its own rows
mine[:, first[rank + 1]:] = np.nan
send = torch.from_numpy(shard.pack_owned(mine, first, rank))
recv = torch.empty(world * send.numel(), dtype=torch.float64)
dist.all_gather_into_tensor(recv, send)                                    # the one exchange step of a sharded matvec
y = shard.unpack_gathered(recv.numpy(), first, perm)
want = np.empty(2 * N); want[perm] = y_morton[0]; want[N + perm] = y_morton[1]
assert not np.isnan(y).any() and np.array_equal(y, want)
# replicated Krylov vectors: the dots need no all-reduce, every rank holds the same full y
t = torch.from_numpy(y.copy()); dist.all_reduce(t, op=dist.ReduceOp.MAX)
assert np.array_equal(t.numpy(), y)
dist.barrier()
if rank == 0:
    print(json.dumps(dict(ok=True, first=[int(f) for f in first], nmax=shard.nmax_of(first))))
dist.destroy_process_group()
"""


def test_sharded_matvec_exchange_layout_gloo_world2(tmp_path):
    script = tmp_path / "shard_worker.py"
    script.write_text(_SHARD_WORKER.format(root=ROOT))
    r = _torchrun([str(script)])
    assert r.returncode == 0, r.stderr[-3000:]
    d = json.loads([l for l in r.stdout.splitlines() if l.startswith("{")][0])
    assert d["ok"] and d["first"][0] == 0 and d["first"][-1] == 1000 and d["first"][1] % 64 == 0
    assert d["nmax"] == max(d["first"][1], 1000 - d["first"][1])
