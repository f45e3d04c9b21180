"""GPU parity of the slab-sharded lattice (include/prs.h "z slabs"; paper_1710_10420_b200/sharded.py).

All slabs of a lattice run on the one GPU of the test box, one after the other (their kernels never
wait on one another; halo planes move by device copies ordered by events).  The bar: after any mix of
step counts the owned planes of the slabs, put together, equal the unsharded lattice BIT FOR BIT (and so
the CPU oracle's FMA form), the link and wall-site counts add up exactly, and the velocity sum agrees to
the rounding of a differently ordered double sum."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import paper_1710_10420_b200 as prs  # noqa: E402
from oracle import binding as ref  # noqa: E402
from paper_1710_10420_b200 import sharded  # noqa: E402

STEPS = [4, 4, 1, 3, 4, 2, 5, 13]          # whole passes, remainders, a fresh halo, a used-up one


def same_diag(a, b):
    assert a["link_count"] == b["link_count"] and a["wall_sites"] == b["wall_sites"], (a, b)
    assert a["step"] == b["step"] and a["eta"] == b["eta"]
    assert abs(a["sum_ratio"] - b["sum_ratio"]) <= 1e-12 * abs(b["sum_ratio"])
    assert abs(a["rho"] - b["rho"]) <= 1e-15 and abs(a["gv2"] - b["gv2"]) <= 1e-12 * abs(b["gv2"])


@pytest.mark.parametrize("N,world", [(4, 1), (8, 2), (12, 3), (20, 5), (64, 1), (64, 2), (64, 4), (64, 16), (132, 3), (128, 8)])
@pytest.mark.parametrize("prec", [prs.F32, prs.F64])
@pytest.mark.parametrize("kernel", [prs.KERNEL_AUTO, prs.KERNEL_GENERIC, "two rows per thread"])
def test_slabs_put_together_equal_the_unsharded_lattice_bitwise(N, world, prec, kernel):
    kw = dict(seed=11, era_m=2.0)
    whole = prs.Simulation(3, N, prec, **kw)
    group = sharded.SlabGroup(N, [0] * world, prec, **kw)
    rows2 = kernel == "two rows per thread"
    if rows2:
        kernel = prs.KERNEL_AUTO
    for s in group.slabs:
        s.set_step_kernel(kernel)
        if rows2:
            s.set_option(8, 2)                                          # PRS_OPT_TBS_ROWS
    whole.init(1.0)
    group.init(1.0)
    wp, wv = whole.copy_out()
    gp, gv = group.copy_out()
    assert gp.tobytes() == wp.tobytes() and gv.tobytes() == wv.tobytes()
    same_diag(group.diagnostics(), whole.diagnostics())
    for k in STEPS:
        whole.step(k)
        group.step(k)
        wp, wv = whole.copy_out()
        gp, gv = group.copy_out()
        assert gp.tobytes() == wp.tobytes() and gv.tobytes() == wv.tobytes(), k
        same_diag(group.diagnostics(), whole.diagnostics())
    if kernel == prs.KERNEL_AUTO:
        assert all(s.get_info(2) in (prs.KERNEL_TBS, prs.KERNEL_TB2, prs.KERNEL_TILED) for s in group.slabs)
    else:
        assert all(s.get_info(2) == prs.KERNEL_GENERIC for s in group.slabs)
    if N <= 64 and world in (1, 4):                # ... and the oracle's FMA form, bit for bit
        r = ref.RefSim(3, N, prec, arith=ref.ARITH_FMA, **kw)
        r.init(1.0)
        r.step(sum(STEPS))
        rp, rv = r.copy_out()
        assert gp.tobytes() == rp.tobytes() and gv.tobytes() == rv.tobytes()
        dr = r.diagnostics()
        dg = group.diagnostics()
        assert dg["link_count"] == dr["link_count"] and dg["wall_sites"] == dr["wall_sites"]
    group.close()
    whole.close()


def binding_step():
    from paper_1710_10420_b200 import prs as binding
    return binding.INFO_STEP


def test_four_step_kernel_is_what_a_whole_pass_on_a_slab_runs():
    g = sharded.SlabGroup(128, [0, 0], prs.F32, seed=3)
    g.init(1.0)
    before = g.kernel_launches
    g.step(8)
    assert g.kernel_launches - before == 2 * 2                         # two passes on each of two slabs
    assert all(s.get_info(2) == prs.KERNEL_TBS for s in g.slabs)
    g.step(3)                                                          # one three-step pass
    assert all(s.get_info(2) == prs.KERNEL_TBS and s.halo_valid == 0 for s in g.slabs)
    g.step(2)                                                          # one two-step pass over all planes
    assert all(s.get_info(2) == prs.KERNEL_TB2 and s.halo_valid == 2 for s in g.slabs)
    g.step(1)
    assert all(s.get_info(2) == prs.KERNEL_TILED and s.halo_valid == 1 for s in g.slabs)
    g.diagnostics()
    assert all(s.get_info(4) == prs.KERNEL_TILED for s in g.slabs)       # the tiled diagnostics kernel on the owned planes
    g.close()


def test_one_rank_of_a_distributed_job_without_peers():
    """ShardedSimulation with world = 1 (its own neighbour; no process group needed)."""
    N = 64
    whole = prs.Simulation(3, N, prs.F64, seed=5)
    one = sharded.ShardedSimulation(N, prs.F64, rank=0, world=1, seed=5)
    whole.init(1.0)
    one.init(1.0)
    whole.step(21)
    one.step(21)
    wp, wv = whole.copy_out()
    gp, gv = one.copy_out()
    assert gp.tobytes() == wp.tobytes() and gv.tobytes() == wv.tobytes()
    same_diag(one.diagnostics(), whole.diagnostics())
    one.close()
    whole.close()


def test_restoring_a_slab_from_a_snapshot():
    N, world = 64, 2
    a = sharded.SlabGroup(N, [0] * world, prs.F32, seed=9)
    a.init(1.0)
    a.step(10)
    b = sharded.SlabGroup(N, [0] * world, prs.F32, seed=12345)
    for sa, sb in zip(a.slabs, b.slabs):
        p, v = sa.copy_out()
        sb.copy_in(p, v, eta0=1.0, step=10)
        assert sb.halo_valid == 0                                       # the halo belongs to no state yet
    a.step(9)
    b.step(9)
    ap, av = a.copy_out()
    bp, bv = b.copy_out()
    assert ap.tobytes() == bp.tobytes() and av.tobytes() == bv.tobytes()
    same_diag(a.diagnostics(), b.diagnostics())
    a.close()
    b.close()


def test_slab_error_paths():
    s = sharded.SlabSimulation(64, 16, 16, prs.F32)
    with pytest.raises(prs.PrsError) as e:
        s.step(1)                                                       # no state yet
    assert e.value.code == 4
    with pytest.raises(prs.PrsError) as e:
        s.halo_regions()
    assert e.value.code == 4
    s.init(1.0)
    assert s.halo_valid == 4
    with pytest.raises(prs.PrsError) as e:
        s.step(5)                                                       # more than the halo is good for
    assert e.value.code == 4
    s.step(4)
    assert s.halo_valid == 0
    with pytest.raises(prs.PrsError) as e:
        s.step(1)
    assert e.value.code == 4
    with pytest.raises(prs.PrsError) as e:
        s.diagnostics()                                                 # stale halo
    assert e.value.code == 4
    with pytest.raises(prs.PrsError) as e:
        s.weighted_area()                                               # stale halo as well
    assert e.value.code == 4
    with pytest.raises(prs.PrsError) as e:
        s.set_step_kernel(prs.KERNEL_TB2)
    assert e.value.code == 2
    s.halo_filled()
    s.step(2)
    assert s.halo_valid == 2 and s.get_info(binding_step()) == 6
    s.halo_filled()
    s.step(3)                                                           # a three-step pass leaves the halo stale
    assert s.halo_valid == 0 and s.get_info(binding_step()) == 9
    s.close()
    for N, z0, nz in ((66, 0, 16), (64, 0, 3), (64, 64, 16), (64, -1, 16), (64, 0, 65)):
        with pytest.raises(prs.PrsError):
            sharded.SlabSimulation(N, z0, nz, prs.F32)
    whole = prs.Simulation(3, 64, prs.F32)
    whole.init(1.0)
    assert whole.get_info(sharded.INFO_HALO_PLANES) == 0
    assert sharded._slab_lib().prs_slab_halo_filled(whole._h) == 4     # PRS_ERR_STATE: not a slab
    whole.close()


def test_eight_slabs_of_512_cubed_match_the_unsharded_lattice():
    """A BASELINE.json lattice (512^3 FP32) as eight slabs of 64 planes: what each of eight GPUs would hold."""
    N, world = 512, 8
    whole = prs.Simulation(3, N, prs.F32, seed=2)
    group = sharded.SlabGroup(N, [0] * world, prs.F32, seed=2)
    whole.init(1.0)
    group.init(1.0)
    whole.step(22)
    group.step(22)
    wp, wv = whole.copy_out()
    gp, gv = group.copy_out()
    assert np.array_equal(gp.view(np.uint32), wp.view(np.uint32)) and np.array_equal(gv.view(np.uint32), wv.view(np.uint32))
    same_diag(group.diagnostics(), whole.diagnostics())
    group.close()
    whole.close()


@pytest.mark.parametrize("N,world,prec", [(128, 4, prs.F32), (96, 3, prs.F64)])
def test_a_long_sharded_run_tracks_the_unsharded_one_exactly(N, world, prec):
    """630 steps (eta 1 -> 64) with diagnostics every 10 steps: ~190 halo exchanges, whole passes and the
    two-step remainder in turn.  The chaotic network amplifies any single wrong halo value within a few
    tens of steps, so identical counts at every sample and identical fields at the end mean every
    exchange put every plane in the right place."""
    whole = prs.Simulation(3, N, prec, seed=4)
    group = sharded.SlabGroup(N, [0] * world, prec, seed=4)
    whole.init(1.0)
    group.init(1.0)
    for _ in range(63):
        whole.step(10)
        group.step(10)
        same_diag(group.diagnostics(), whole.diagnostics())
    wp, wv = whole.copy_out()
    gp, gv = group.copy_out()
    assert gp.tobytes() == wp.tobytes() and gv.tobytes() == wv.tobytes()
    d = group.diagnostics()
    assert 0 < d["link_count"] < 0.2 * N ** 3                            # a network has formed
    group.close()
    whole.close()


RANK_WORKER = r"""
import os, sys
sys.path.insert(0, %r)
import numpy as np
import torch
import torch.distributed as dist
import paper_1710_10420_b200 as prs
from paper_1710_10420_b200 import sharded
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
torch.cuda.set_device(0)
dist.init_process_group("gloo")
sim = sharded.ShardedSimulation(%d, prs.F32, seed=5, era_m=2.0)
sim.init(1.0)
diags = []
areas = []
for k in (4, 9, 2, 6):
    sim.step(k)
    diags.append(sim.diagnostics())
    areas.append(sim.weighted_area()[0])           # the slabs' partial areas, all-reduced over the ranks
phi, pd = sim.copy_out()
np.save(os.path.join(%r, "phi%%d.npy" %% rank), phi)
np.save(os.path.join(%r, "pd%%d.npy" %% rank), pd)
np.save(os.path.join(%r, "diag%%d.npy" %% rank), np.array([[d["link_count"], d["wall_sites"], d["sum_ratio"], a] for d, a in zip(diags, areas)]))
dist.barrier()
sim.close()
dist.destroy_process_group()
"""


@pytest.mark.parametrize("world", [2, 3])
def test_ranks_of_a_distributed_job_share_the_one_gpu(world, tmp_path):
    """ShardedSimulation as torchrun would start it, one process per rank, all on cuda:0, halo planes and
    the diagnostics sums over torch.distributed (gloo; blocks staged through the host).  Processes take
    turns on the GPU; no kernel waits on another."""
    import os
    import subprocess
    import sys

    from tests.test_bench_replicas_cpu import free_port

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    N, port, out = 48, free_port(), str(tmp_path)
    procs = []
    for rank in range(world):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", RANK_WORKER % (root, N, out, out, out)], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=600) for p in procs]
    assert [p.returncode for p in procs] == [0] * world, outs
    whole = prs.Simulation(3, N, prs.F32, seed=5, era_m=2.0)
    whole.init(1.0)
    want = []
    for k in (4, 9, 2, 6):
        whole.step(k)
        d = whole.diagnostics()
        want.append([d["link_count"], d["wall_sites"], d["sum_ratio"], whole.weighted_area()[0]])
    wp, wv = whole.copy_out()
    whole.close()
    gp = np.concatenate([np.load(os.path.join(out, "phi%d.npy" % r)) for r in range(world)])
    gv = np.concatenate([np.load(os.path.join(out, "pd%d.npy" % r)) for r in range(world)])
    assert gp.tobytes() == wp.tobytes() and gv.tobytes() == wv.tobytes()
    want = np.array(want)
    for r in range(world):                                               # every rank holds the lattice's sums
        got = np.load(os.path.join(out, "diag%d.npy" % r))
        assert np.array_equal(got[:, :2], want[:, :2])
        assert np.allclose(got[:, 2], want[:, 2], rtol=1e-12, atol=0)
        assert np.allclose(got[:, 3], want[:, 3], rtol=1e-12, atol=0)       # Eq. 7's weighted area of the whole lattice


@pytest.mark.parametrize("N,world", [(64, 1), (64, 4), (132, 3), (256, 2)])        # 256^3 in two slabs: the sign-bit path
@pytest.mark.parametrize("prec", [prs.F32, prs.F64])
def test_weighted_area_of_the_slabs_adds_up_to_the_lattice(N, world, prec):
    """prs_weighted_area on a slab returns its partial sum of Eq. 7's weighted area (transverse neighbours of the
    links of the outermost owned planes are halo planes); the parts add up to the unsharded lattice's and to the
    oracle's value on the same bytes, on the initial field and on a formed network, with a fresh and a used halo."""
    whole = prs.Simulation(3, N, prec, seed=4)
    group = sharded.SlabGroup(N, [0] * world, prec, seed=4)
    whole.init(1.0)
    group.init(1.0)
    for k in (0, 4, 3, 60, 1):
        whole.step(k)
        group.step(k)
        a_w, r_w = whole.weighted_area()
        a_g, r_g = group.weighted_area()
        want = ref.weighted_area_of(whole.copy_out()[0])
        assert abs(a_g - a_w) <= 1e-12 * max(a_w, 1.0) and abs(a_g - want) <= 1e-12 * max(want, 1.0)
        assert abs(r_g - r_w) <= 1e-15
    s = group.slabs[0]
    s.step(s.halo_valid)                                      # use the halo up: the call must refuse, not misread
    if world > 1:
        with pytest.raises(prs.PrsError):
            s.weighted_area()
    group.close()
    whole.close()


def test_sharded_simulation_on_a_stream_of_its_own():
    """The halo transport must run on the slab's stream: with a non-default, non-blocking stream the
    copies would otherwise race with the step kernels.  world = 1: the slab is its own neighbour."""
    import torch

    N = 96
    st = torch.cuda.Stream()
    whole = prs.Simulation(3, N, prs.F32, seed=5)
    one = sharded.ShardedSimulation(N, prs.F32, rank=0, world=1, seed=5, stream=st)
    whole.init(1.0)
    one.init(1.0)
    for k in (4, 4, 4, 9, 2):
        whole.step(k)
        one.step(k)
    one.slab.sync()
    wp, wv = whole.copy_out()
    gp, gv = one.copy_out()
    assert gp.tobytes() == wp.tobytes() and gv.tobytes() == wv.tobytes()
    same_diag(one.diagnostics(), whole.diagnostics())
    assert abs(one.weighted_area()[0] - whole.weighted_area()[0]) <= 1e-12 * whole.weighted_area()[0]
    one.close()
    whole.close()


def test_handles_work_whatever_device_is_current():
    """A handle belongs to the device that owns its workspace (include/prs.h "Devices"): every call switches to it
    and restores the caller's device.  With one GPU this checks the restore; with two or more, that a handle on
    device 1 can be driven while device 0 is current and that the > 48 KB shared-memory attribute is set per device."""
    import torch
    from paper_1710_10420_b200 import prs as binding

    ndev = torch.cuda.device_count()
    dev = ndev - 1
    with torch.cuda.device(dev):
        g = prs.Simulation(3, 128, prs.F32, seed=7)            # 128^3: the four-step kernel (172 KB of shared memory)
    assert g.get_info(binding.INFO_DEVICE) == dev
    torch.cuda.set_device(0)
    g.init(1.0)
    g.step(9)
    d = g.diagnostics()
    assert torch.cuda.current_device() == 0
    assert g.get_info(binding.INFO_STEP_KERNEL) == prs.KERNEL_TBS
    ref_g = prs.Simulation(3, 128, prs.F32, seed=7)            # on device 0
    ref_g.init(1.0)
    ref_g.step(9)
    same_diag(d, ref_g.diagnostics())
    assert g.copy_out()[0].tobytes() == ref_g.copy_out()[0].tobytes()
    g.close()
    ref_g.close()


def test_slab_group_over_two_devices():
    import torch

    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs in one process (the box has one); see test_handles_work_whatever_device_is_current")
    N = 128
    whole = prs.Simulation(3, N, prs.F32, seed=3)
    group = sharded.SlabGroup(N, [0, 1], prs.F32, seed=3)
    whole.init(1.0)
    group.init(1.0)
    for k in STEPS:
        whole.step(k)
        group.step(k)
        wp, wv = whole.copy_out()
        gp, gv = group.copy_out()
        assert gp.tobytes() == wp.tobytes() and gv.tobytes() == wv.tobytes(), k
        same_diag(group.diagnostics(), whole.diagnostics())
    group.close()
    whole.close()


@pytest.mark.parametrize("N,world", [(128, 1), (128, 4), (256, 8)])
@pytest.mark.parametrize("prec", [prs.F32, prs.F64])
def test_sign_bit_diagnostics_on_slabs(N, world, prec):
    """The packed-sign-bit diagnostics pass (PRS_KERNEL_BITS) on z slabs: a slab packs the signs of its owned planes and
    of one halo plane on either side and measures the owned planes; the parts add up to the unsharded lattice's."""
    from paper_1710_10420_b200 import prs as binding

    whole = prs.Simulation(3, N, prec, seed=6)
    group = sharded.SlabGroup(N, [0] * world, prec, seed=6)
    for s in group.slabs:
        s.set_option(binding.OPT_DIAG_KERNEL, prs.KERNEL_BITS)
    whole.set_option(binding.OPT_DIAG_KERNEL, prs.KERNEL_TILED)
    whole.init(1.0)
    group.init(1.0)
    for k in (0, 4, 3, 120, 1):
        whole.step(k)
        group.step(k)
        same_diag(group.diagnostics(), whole.diagnostics())
        assert all(s.get_info(4) == prs.KERNEL_BITS for s in group.slabs)
    group.close()
    whole.close()
