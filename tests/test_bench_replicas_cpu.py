"""Multi-GPU leg of bench.py on the CPU (gloo, world_size 2): the path does not shard (DESIGN.md section 7,
"replicas only"), so the only cross-rank logic is the aggregation -- MAX of the times, SUM of the counts,
whole-job throughput -- and the rule that rank 0 alone prints.  No GPU, no libprs call."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, %r)
import torch.distributed as dist
import bench
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
times, counts = bench.reduce_over_ranks([10.0 + 5.0 * rank, 3.0 - rank], [7 + rank], world, "cpu")
value = bench.aggregate_value(1000, 50, 2, world, times[0])
dist.barrier()
if rank == 0:
    print(json.dumps({"times": times, "counts": counts, "value": value}))
dist.destroy_process_group()
"""


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_replicas_aggregate_like_the_bench_contract_says():
    port = free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER % ROOT], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=300) for p in procs]
    assert [p.returncode for p in procs] == [0, 0], outs
    assert outs[1][0].strip() == ""                        # only rank 0 prints
    got = json.loads(outs[0][0].strip().splitlines()[-1])
    assert got["times"] == [15.0, 3.0]                     # max over ranks
    assert got["counts"] == [15]                           # 7 + 8
    assert got["value"] == 1000 * 50 * 2 * 2 / 15.0e-3     # both replicas' work over the slowest rank's time


def test_single_process_is_a_no_op():
    sys.path.insert(0, ROOT)
    import bench

    assert bench.reduce_over_ranks([1.5, 2.5], [3], 1) == ([1.5, 2.5], [3])
    assert bench.aggregate_value(10, 5, 2, 1, 1000.0) == 100.0


def test_reference_arm_prints_on_rank_zero_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--steps", "1", "--warmup", "0"], env=env, stdout=subprocess.PIPE, text=True, timeout=300)
    assert out.returncode == 0 and out.stdout.strip() == ""
