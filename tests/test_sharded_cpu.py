"""Host logic of the slab-sharded lattice (paper_1710_10420_b200/sharded.py) without a GPU: slab bounds,
the step / exchange schedule, the sum of the slabs' diagnostics, and the halo transport over
torch.distributed with the gloo backend (world sizes 2 and 3) on CPU tensors that stand in for the slabs'
workspaces.  Every plane carries its global plane number, so a block that lands in the wrong halo, or
from the wrong neighbour, or in the wrong order, shows.  No libprs compute call here; the kernels on
slabs are covered by tests/test_gpu_parity.py (-m gpu)."""
import json
import os
import subprocess
import sys

import pytest

from paper_1710_10420_b200 import sharded
from tests.test_bench_replicas_cpu import free_port

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_slab_bounds_cover_the_lattice_once():
    for N, world in ((64, 1), (64, 2), (64, 4), (64, 16), (1024, 8)):
        got = [sharded.slab_bounds(N, world, r) for r in range(world)]
        assert [b for b, _ in got] == [r * (N // world) for r in range(world)]
        assert sum(n for _, n in got) == N
    for N, world in ((64, 3), (64, 32), (12, 4)):                  # uneven, or slabs thinner than the halo
        with pytest.raises(ValueError):
            sharded.slab_bounds(N, world, 0)
    with pytest.raises(ValueError):
        sharded.slab_bounds(64, 2, 2)


def test_step_schedule_never_outruns_the_halo():
    for nsteps in range(0, 23):
        for valid in range(0, 5):
            ops = sharded.step_schedule(nsteps, valid)
            v, done = valid, 0
            for op in ops:
                if op[0] == "exchange":
                    assert v < sharded.HALO                        # never exchanges a fresh halo
                    v = sharded.HALO
                else:
                    assert 1 <= op[1] <= min(sharded.HALO, v)      # a step never outruns the halo
                    v -= op[1]
                    done += op[1]
            assert done == nsteps
            # whole passes of four first, one remainder at the end
            ks = [op[1] for op in ops if op[0] == "step"]
            assert all(k == 4 for k in ks[:-1])
    assert sharded.step_schedule(8, 4) == [("step", 4), ("exchange",), ("step", 4)]
    assert sharded.step_schedule(0, 0) == []


def test_combined_diagnostics_are_the_sums():
    parts = [{"step": 7, "eta": 1.7, "link_count": 10, "wall_sites": 4, "sum_ratio": 1.5},
             {"step": 7, "eta": 1.7, "link_count": 2 ** 40, "wall_sites": 6, "sum_ratio": 2.5}]
    d = sharded.combine_diagnostics(parts, 8)
    assert d["link_count"] == 10 + 2 ** 40 and d["wall_sites"] == 10 and d["sum_ratio"] == 4.0
    assert d["rho"] == (10 + 2 ** 40) / 512.0 and d["gv2"] == 4.0 / 20.0 and d["step"] == 7
    assert sharded.combine_diagnostics([dict(parts[0], wall_sites=0, sum_ratio=0.0)], 8)["gv2"] == 0.0


WORKER = r"""
import json, os, sys
sys.path.insert(0, %r)
import torch
import torch.distributed as dist
from paper_1710_10420_b200 import sharded
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
N, H, PL = 24, sharded.HALO, 5                      # PL values per plane stand in for N*N
z0, nz = sharded.slab_bounds(N, world, rank)
# two fields, each (nz + 2H) planes; owned plane l holds 1000*field + global z; halos start as -1
fields = []
for f in range(2):
    a = torch.full((nz + 2 * H, PL), -1.0)
    for l in range(nz):
        a[H + l] = 1000.0 * f + (z0 + l)
    fields.append(a)
send, recv = [], []
for a in fields:
    send += [a[H:2 * H], a[nz:nz + H]]              # lowest / highest owned planes
    recv += [a[0:H], a[H + nz:]]                    # lower / upper halo
sharded.exchange_halo_tensors(send, recv, rank, world)
out = [[int(a[l, 0]) for l in range(nz + 2 * H)] for a in fields]
same = all(bool((a == a[:, :1]).all()) for a in fields)
dist.barrier()
print(json.dumps({"rank": rank, "z0": z0, "nz": nz, "planes": out, "rows_uniform": same}))
dist.destroy_process_group()
"""


@pytest.mark.parametrize("world", [2, 3])
def test_halo_transport_over_gloo_puts_the_right_global_planes_in_every_halo(world):
    port = free_port()
    procs = []
    for rank in range(world):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER % ROOT], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=300) for p in procs]
    assert [p.returncode for p in procs] == [0] * world, outs
    N, H = 24, sharded.HALO
    for rank, (so, _) in enumerate(outs):
        got = json.loads(so.strip().splitlines()[-1])
        assert got["rank"] == rank and got["rows_uniform"]
        for f in range(2):
            want = [1000 * f + (got["z0"] - H + l) % N for l in range(got["nz"] + 2 * H)]
            assert got["planes"][f] == want, (rank, f)


def test_one_slab_is_its_own_neighbour():
    import torch

    H = sharded.HALO
    a = torch.arange(-H, 16 + H, dtype=torch.float64).remainder(16).reshape(-1, 1).clone()   # already right
    b = a.clone()
    b[:H] = -1.0
    b[-H:] = -1.0
    sharded.exchange_halo_tensors([b[H:2 * H], b[16:16 + H]], [b[:H], b[H + 16:]], 0, 1)
    assert torch.equal(a, b)
