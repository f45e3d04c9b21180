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


def test_reference_arm_line_on_a_small_config():
    """--impl reference times the oracle on the workload's own lattice and prints the contract's keys."""
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "2d_256_f32_rad",
                          "--steps", "2", "--warmup", "1"], stdout=subprocess.PIPE, text=True, timeout=300)
    assert out.returncode == 0
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "site_updates_per_sec" and line["value"] > 0
    assert line["config"]["workload"] == "2d_256_f32_rad" and line["config"]["N"] == 256
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["value"] == line["value"]
    assert line["e2e"] == {"value": line["value"], "unit": line["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert "256^2" in line["cpu_baseline"]["sample"]


def test_ncu_traffic_is_reported_only_for_the_kernel_that_was_launched(tmp_path, monkeypatch):
    sys.path.insert(0, ROOT)
    import bench

    rec = {"captures": [{"profile": "x.md", "kernel": "step3d_tbr_kernel<float,2,4,24,1>", "grid": [9, 43, 8],
                         "block": [32, 16, 1], "dram_bytes_read": 10, "dram_bytes_write": 5}]}
    f = tmp_path / "ncu_traffic.json"
    f.write_text(json.dumps(rec))
    monkeypatch.setattr(bench, "NCU_TRAFFIC_FILE", str(f))
    hit = {"kernel": "step3d_tbr_kernel<float,2,4,24,1>", "grid": [9, 43, 8], "block": [32, 16, 1]}
    assert bench.ncu_traffic_for(hit)[0] == 15
    for miss in (dict(hit, kernel="step3d_tbr_kernel<float,2,4,24,0>"), dict(hit, grid=[9, 43, 4]), dict(hit, block=[32, 24, 1])):
        got, why = bench.ncu_traffic_for(miss)
        assert got is None and "no committed ncu capture" in why
    # the committed record parses and every entry names its profile summary, which exists
    monkeypatch.undo()
    if os.path.exists(bench.NCU_TRAFFIC_FILE):
        for c in json.load(open(bench.NCU_TRAFFIC_FILE))["captures"]:
            assert os.path.exists(os.path.join(ROOT, "profiles", c["profile"])), c["profile"]
            assert len(c["grid"]) == 3 and len(c["block"]) == 3 and c["dram_bytes_read"] > 0
