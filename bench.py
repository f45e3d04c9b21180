#!/usr/bin/env python
"""bench.py -- headline benchmark of the PRS hot path (BASELINE.json: site-updates/s and achieved HBM
GB/s, 3D 1024^3 FP32).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config NAME]

One bench "step" is one pass of the whole hot path over the resident lattice: SUBSTEPS fused PRS
steps (Eqs. 3-6, prs_step) followed by one diagnostics pass (Eqs. 7-8, prs_diagnostics:
link count, wall sites, velocity sum, 24-byte readback).  SUBSTEPS = 50 is the diagnostics cadence of
BASELINE.json's 3D configs.  `value` = site-updates per second with the state resident in HBM; `e2e`
is the same cycle driven through the C ABI with HOST buffers: prs_copy_in from pinned host memory,
the same SUBSTEPS + diagnostics, prs_copy_out back to pinned host memory, all inside the timed region.

Multi-GPU: the path does not shard under north_star ("one GPU, no sharding, no collectives"), so
--gpus N runs N independent replicas (different seeds, the paper's multi-seed ensemble)
and reports the aggregate: "scaling": "weak".  There is no data-path collective; torch.distributed is
used only for the barrier and the max-over-ranks of the device time.

--impl reference times the CPU oracle (oracle/, plain C++ restatement of the paper's equations) on
the host cores on a bounded sample of the same workload.  It is a deliberately slow program: a
reported baseline, not the target.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "site_updates_per_sec"
UNIT = "site-updates/s"
SUBSTEPS = 50

# name -> (dims, N, precision, era_m); precision 0 = FP32, 1 = FP64.  Parameters common to all
# BASELINE.json configs: alpha=3, deta=0.1, W0=10, phi0=1, eta0=1, seeded uniform(-1,1) init.
CONFIGS = {
    "3d_1024_f32_rad": (3, 1024, 0, 1.0),      # headline (BASELINE.json metric; configs[4])
    "3d_1024_f32_mat": (3, 1024, 0, 2.0),
    "3d_1024_f64_rad": (3, 1024, 1, 1.0),
    "3d_512_f32_rad": (3, 512, 0, 1.0),        # configs[3]
    "2d_16384_f32_rad": (2, 16384, 0, 1.0),    # configs[2]
    "2d_16384_f64_rad": (2, 16384, 1, 1.0),
    "2d_4096_f32_rad": (2, 4096, 0, 1.0),      # configs[1]
    "2d_4096_f32_mat": (2, 4096, 0, 2.0),
    "2d_256_f32_rad": (2, 256, 0, 1.0),        # configs[0]
}
# diagnostics cadence BASELINE.json states for the small config ("wall link-count every 10 steps")
OWN_CADENCE = {"2d_256_f32_rad": 10}
DEFAULT_CONFIG = "3d_1024_f32_rad"
BYTES_PER_SITE_UPDATE = {0: 16, 1: 32}        # read phi, phidot; write phidot, phi

NCU_TRAFFIC_FILE = os.path.join(ROOT, "profiles", "ncu_traffic.json")


def ensemble_leg(prs, torch, stream, dims, N, prec, era_m, ncyc, cad, sites, boxes=16):
    """`boxes` independent lattices (seeds 101...) advanced side by side: prs_run(ncyc, cad) from one host thread per
    handle, each handle on a stream of its own.  Device time from a start event every stream waits for to the last
    stream's end event."""
    import threading

    streams = [torch.cuda.Stream() for _ in range(boxes)]
    sims = [prs.Simulation(dims, N, prec, era_m=era_m, seed=101 + i, stream=streams[i]) for i in range(boxes)]
    try:
        for sm in sims:
            sm.init(1.0)
            sm.run(2, cad)                                           # warm-up (and the per-device kernel attributes)
        torch.cuda.synchronize()
        errors = []

        def drive(sm):
            try:
                sm.run(ncyc, cad)
            except Exception as exc:                                 # surfaces below
                errors.append(exc)

        start = torch.cuda.Event(enable_timing=True)
        start.record(stream)
        for st in streams:
            st.wait_event(start)
        threads = [threading.Thread(target=drive, args=(sm,)) for sm in sims]
        for t in threads:
            t.start()
        for t in threads:
            t.join()
        ends = []
        for st in streams:
            e = torch.cuda.Event(enable_timing=True)
            e.record(st)
            ends.append(e)
        torch.cuda.synchronize()
        if errors:
            raise errors[0]
        ms = max(start.elapsed_time(e) for e in ends)
        box_steps = boxes * ncyc * cad
        return {"boxes": boxes, "cycle": "%d PRS steps + 1 diagnostics pass, %d cycles per box" % (cad, ncyc),
                "us_per_box_step": ms * 1e3 / box_steps, "box_steps_per_s": box_steps / ms * 1e3,
                "site_updates_per_s": box_steps * sites / ms * 1e3, "step_kernel": sims[0].step_launch_info()["kernel"]}
    finally:
        for sm in sims:
            sm.close()


def ncu_traffic_for(launch):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the kernel that was ACTUALLY launched, from
    the committed record of `ncu --set full` captures (profiles/ncu_traffic.json: one entry per capture with the
    kernel's name and template arguments, grid, block and bytes).  A capture counts only if kernel, grid and
    block all equal what prs_step_launch_info reports for this run; otherwise (None, why)."""
    try:
        with open(NCU_TRAFFIC_FILE) as fh:
            captures = json.load(fh)["captures"]
    except Exception as exc:
        return None, "no capture record (%s)" % exc
    for c in captures:
        if c["kernel"] == launch["kernel"] and c["grid"] == launch["grid"] and c["block"] == launch["block"]:
            return (int(c["dram_bytes_read"]) + int(c["dram_bytes_write"]),
                    "ncu capture %s" % c["profile"] + ("; " + c["note"] if c.get("note") else ""))
    return None, "no committed ncu capture of %s grid %s block %s" % (launch["kernel"], launch["grid"], launch["block"])


def measured_peak_gbs():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons for one GPU while the timed region runs."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.t.join(timeout=5)
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); power.append(float(r[2]))
            except ValueError:
                continue
            for name, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def host_threads():
    try:
        return len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count() or 1


def oracle_sample(dims, prec, era_m, nsteps, threads, N, seed=1):
    """Times the oracle as it stands on `threads` host threads on the workload's own lattice: seeded init
    (untimed), `nsteps` PRS steps, one diagnostics pass.  Returns a dict with the times and the metric at the
    bench's cadence: SUBSTEPS steps + 1 diagnostics pass per cycle, i.e. value = SUBSTEPS N^d /
    (SUBSTEPS t_step + t_diag) -- the same quantity the GPU arm reports, from a bounded sample of the cycle."""
    from oracle import binding as ref

    sim = ref.RefSim(dims, N, prec, era_m=era_m, seed=seed, threads=threads)
    t0 = time.perf_counter()
    sim.init(1.0)
    t1 = time.perf_counter()
    sim.step(nsteps)
    t2 = time.perf_counter()
    d = sim.diagnostics()
    t3 = time.perf_counter()
    sim.close()
    t_step, t_diag = (t2 - t1) / nsteps, t3 - t2
    S = N ** dims
    return {"N": N, "nsteps": nsteps, "t_init_s": t1 - t0, "t_step_s": t_step, "t_diag_s": t_diag,
            "value": SUBSTEPS * S / (SUBSTEPS * t_step + t_diag), "steps_only_value": S / t_step,
            "desc": "%dD %d^%d %s (the workload's own lattice), oracle as it stands on %d thread(s): %d PRS steps timed "
                    "(%.2f s each) + 1 diagnostics pass (%.2f s, on the state after those steps); value = %d N^d / (%d t_step + t_diag), "
                    "the bench cycle's cadence; seeded init %.1f s not timed; rho=%.5f"
                    % (dims, N, dims, "FP32" if prec == 0 else "FP64", threads, nsteps, t_step, t_diag, SUBSTEPS, SUBSTEPS,
                       t1 - t0, d["rho"])}


def reduce_over_ranks(times_ms, counts, world, device="cpu"):
    """Replica aggregation: a job is as slow as its slowest rank, so every time
    is the MAX over ranks; counts (kernel launches) are SUMmed.  No data-path collective: these few
    scalars are the only thing the ranks ever exchange.  Works on any backend (nccl on the GPUs,
    gloo in the CPU test)."""
    if world <= 1:
        return [float(t) for t in times_ms], [int(c) for c in counts]
    import torch
    import torch.distributed as dist

    t = torch.tensor([float(x) for x in times_ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor([int(x) for x in counts], device=device, dtype=torch.int64)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return [float(x) for x in t.tolist()], [int(x) for x in c.tolist()]


def aggregate_value(sites, substeps, steps, world, ms_total):
    """Whole-job site-updates per second of `world` replicas that each did steps x substeps PRS steps."""
    return sites * substeps * steps * world / (ms_total * 1e-3)


def run_reference(args):
    """--impl reference: the oracle on the host cores, on this arm's config, metric and unit.  One bench step = a
    bounded sample of the cycle on the workload's own lattice: 2 PRS steps timed; the diagnostics pass is timed
    once (in the warm-up) and enters every step's value at the cycle's cadence."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    dims, N, prec, era_m = CONFIGS[args.config]
    threads = host_threads()
    from oracle import binding as ref

    S = N ** dims
    nsub = 2
    sim = ref.RefSim(dims, N, prec, era_m=era_m, seed=1, threads=threads)
    t0 = time.perf_counter()
    sim.init(1.0)
    t_init = time.perf_counter() - t0
    for _ in range(max(1, min(args.warmup, 1))):                 # one warm pass is enough for a CPU loop
        sim.step(1)
    t0 = time.perf_counter()
    d = sim.diagnostics()
    t_diag = time.perf_counter() - t0
    t_steps = []
    for _ in range(args.steps):
        t0 = time.perf_counter()
        sim.step(nsub)
        t_steps.append((time.perf_counter() - t0) / nsub)
    sim.close()
    t_step = sum(t_steps) / len(t_steps)
    t_cycle = SUBSTEPS * t_step + t_diag
    value = SUBSTEPS * S / t_cycle
    desc = ("%dD %d^%d %s (the workload's own lattice), oracle as it stands on %d threads; per bench step %d PRS steps "
            "timed (mean %.2f s per PRS step), diagnostics pass timed once (%.2f s); value = %d N^d / (%d t_step + t_diag) "
            "(the cycle's cadence); seeded init %.1f s not timed; rho=%.5f"
            % (dims, N, dims, "FP32" if prec == 0 else "FP64", threads, nsub, t_step, t_diag, SUBSTEPS, SUBSTEPS, t_init, d["rho"]))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_cycle,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if prec == 0 else "f64", "data": "synthetic",
        "config": {"workload": args.config, "dims": dims, "N": N, "era_m": era_m, "alpha": 3.0, "deta": 0.1,
                   "W0": 10.0, "substeps_per_step": SUBSTEPS, "diagnostics_per_step": 1,
                   "note": "ms_per_step = one cycle of %d PRS steps + 1 diagnostics pass, extrapolated from the timed sample "
                           "(cpu_baseline.sample)" % SUBSTEPS},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def run_gpu(args):
    import torch
    import torch.distributed as dist

    import paper_1710_10420_b200 as prs
    from paper_1710_10420_b200 import prs as binding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the product has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    dims, N, prec, era_m = CONFIGS[args.config]
    S = N ** dims
    bpu = BYTES_PER_SITE_UPDATE[prec]
    slabs = args.decomposition == "slabs"
    if slabs:
        # Opt-in: ONE lattice as z slabs -- under torchrun one slab per rank, halo planes
        # over NCCL ("strong" scaling); in a single process --slabs R slabs one after the other on this GPU,
        # halo planes by device copies: what each of R GPUs would compute, without the NVLink transport.
        from paper_1710_10420_b200 import sharded

        if dims != 3:
            raise SystemExit("--decomposition slabs is for the 3D configs")
        if world > 1:
            sim = sharded.ShardedSimulation(N, prec, rank=rank, world=world, era_m=era_m, seed=1)
        else:
            sim = sharded.SlabGroup(N, [local] * args.slabs, prec, era_m=era_m, seed=1)
        sim.init(1.0)
        stream = torch.cuda.current_stream()
        for _ in range(args.warmup):
            sim.step(SUBSTEPS)
            sim.diagnostics()
        sampler = ClockSampler(local)
        if rank == 0:
            sampler.start()
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0 = sim.kernel_launches
        barrier()
        t0.record(stream)
        for _ in range(args.steps):
            sim.step(SUBSTEPS)
            diag = sim.diagnostics()
        t1.record(stream)
        barrier()
        clocks = sampler.stop() if rank == 0 else None
        (ms_total,), (launches,) = reduce_over_ranks([t0.elapsed_time(t1)], [sim.kernel_launches - l0], world, "cuda")
        value = S * SUBSTEPS * args.steps / (ms_total * 1e-3)          # one lattice, whatever the number of slabs
        peak, peak_src = measured_peak_gbs()
        if rank == 0:
            print(json.dumps({
                "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
                "dtype": "f32" if prec == 0 else "f64", "data": "synthetic",
                "config": {"workload": args.config, "dims": dims, "N": N, "era_m": era_m, "substeps_per_step": SUBSTEPS,
                           "diagnostics_per_step": 1,
                           "parallelism": ("z slabs x%d, one per GPU, halo planes over NCCL" % world) if world > 1
                           else ("z slabs x%d on one GPU one after the other, halo planes by device copies" % args.slabs),
                           "l2": "state exceeds L2; no flush needed"},
                "roofline": {"bound": "hbm", "achieved": value * bpu / 1e9, "peak": peak * world, "unit": "GB/s",
                             "frac": value * bpu / 1e9 / (peak * world), "traffic": None, "peak_source": peak_src,
                             "kernel": "whole cycle (steps, halo transport, diagnostics)"},
                "cpu_baseline": None, "e2e": None, "gpu_launches": launches, "clocks": clocks,
                "last_diag": {k: diag[k] for k in ("step", "eta", "link_count", "wall_sites", "rho", "gv2")}}))
        sim.close()
        if world > 1:
            dist.destroy_process_group()
        return 0
    leg = time_leg(args, args.config, args.steps, args.warmup, world, rank, local, barrier, with_e2e=True, sample_clocks=True)

    # ---- the other precision of BASELINE.json's metric ("3D 1024^3 FP32/FP64"): a short FP64 leg of the same workload,
    # its own events and roofline, outside the FP32 timed region
    also = None
    if args.config == DEFAULT_CONFIG and not args.no_also:
        try:
            other = time_leg(args, "3d_1024_f64_rad", max(2, min(args.steps, 3)), 3, world, rank, local, barrier,
                             with_e2e=False, sample_clocks=False)
            also = {"3d_1024_f64_rad": {k: other[k] for k in ("value", "unit", "dtype", "steps", "warmup", "ms_per_step",
                                                                "roofline", "gpu_launches", "last_diag")}}
        except Exception as exc:
            also = {"3d_1024_f64_rad": {"error": str(exc)[:200]}}
        # ---- and BASELINE.json's configs[0] (2D 256^2 FP32, diagnostics every 10 steps): launch- and latency-bound, so what
        # counts is microseconds per PRS step of the whole cycle (small_lattice), not an HBM fraction
        try:
            tiny = time_leg(args, "2d_256_f32_rad", 3, 3, world, rank, local, barrier, with_e2e=False, sample_clocks=False)
            also["2d_256_f32_rad"] = {k: tiny[k] for k in ("value", "unit", "dtype", "steps", "warmup", "ms_per_step",
                                                            "gpu_launches", "last_diag", "small_lattice")}
            also["2d_256_f32_rad"]["step_kernel"] = tiny["roofline"]["kernel"]
        except Exception as exc:
            also["2d_256_f32_rad"] = {"error": str(exc)[:200]}

    # ---- oracle on the host cores, rank 0, N=1 only: the workload's own lattice, the cycle's cadence
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        threads = host_threads()
        o = oracle_sample(dims, prec, era_m, 2, threads, N)
        o1 = oracle_sample(dims, prec, era_m, 2, 1, 256 if dims == 3 else 4096)
        cpu = {"value": o["value"], "unit": UNIT, "cores": threads, "kind": "oracle", "sample": o["desc"],
               "steps_only_value": o["steps_only_value"],
               "single_thread_value": o1["value"], "single_thread_sample": o1["desc"]}

    if rank == 0:
        line = {
            "metric": METRIC, "value": leg["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": leg["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": leg["dtype"], "data": "synthetic",
            "config": leg["config"], "roofline": leg["roofline"], "cpu_baseline": cpu, "e2e": leg["e2e"],
            "gpu_launches": leg["gpu_launches"], "clocks": leg["clocks"], "last_diag": leg["last_diag"], "also": also,
            "small_lattice": leg["small_lattice"],
        }
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def time_leg(args, config, steps, warmup, world, rank, local, barrier, with_e2e, sample_clocks):
    """One workload: W untimed cycles, then exactly K timed ones (device clock, max over ranks), the step kernel's
    own events, optionally the end-to-end cycle with host buffers.  One cycle = SUBSTEPS PRS steps + 1 diagnostics pass."""
    import torch

    import paper_1710_10420_b200 as prs
    from paper_1710_10420_b200 import prs as binding

    dims, N, prec, era_m = CONFIGS[config]
    S = N ** dims
    bpu = BYTES_PER_SITE_UPDATE[prec]
    sim = prs.Simulation(dims, N, prec, era_m=era_m, seed=rank + 1)
    if args.kernel:
        sim.set_step_kernel({"generic": prs.KERNEL_GENERIC, "tiled": prs.KERNEL_TILED, "tb2": prs.KERNEL_TB2,
                             "tbs": prs.KERNEL_TBS}[args.kernel])
    if args.tbs_rows:
        sim.set_option(binding.OPT_TBS_ROWS, args.tbs_rows)
    if args.tbs_loader:
        sim.set_option(binding.OPT_TBS_LOADER, args.tbs_loader)
    sim.init(1.0)
    stream = torch.cuda.current_stream()
    # what prs_step(SUBSTEPS) launches first is its main kernel; the cycle is issued as prs_step(main) + prs_step(rest)
    # so that the main kernel's launches -- and nothing else -- sit between their own pair of events
    sim.step(SUBSTEPS)
    info = sim.step_launch_info()
    spl = info["steps_per_launch"]
    main_steps = (SUBSTEPS // spl) * spl
    if SUBSTEPS - main_steps == 2 and main_steps >= 2 * spl and (
            (dims == 2 and ((prec == 0 and spl == 8) or (prec == 1 and spl == 6))) or (dims == 3 and spl == 4)):
        # prs_step(50) is 5 x 8 + 6 + 4 steps in 2D FP32, 7 x 6 + 8 in 2D FP64 and 11 x 4 + 3 + 3 in 3D (prs_api.cu: a
        # remainder of 2 trades the last 8 + 2 for 6 + 4, the last 6 + 2 for one 8, the last 4 + 2 for 3 + 3): the second
        # call must see that last main launch to schedule the cycle the way one call would
        main_steps -= spl
    main_launches = main_steps // spl

    def hot_path(ev=None):
        if ev:
            ev[0].record(stream)
        sim.step(main_steps)
        if ev:
            ev[1].record(stream)
        if SUBSTEPS > main_steps:
            sim.step(SUBSTEPS - main_steps)
        return sim.diagnostics()

    sim.diagnostics()
    for _ in range(max(0, warmup - 1)):
        hot_path()
    sim.step(main_steps)
    launch = sim.step_launch_info()                              # the kernel the timed region launches
    sim.step(SUBSTEPS - main_steps)
    sim.diagnostics()
    # ---- timed region: exactly K cycles, device clock, max over ranks
    sampler = ClockSampler(local)
    if rank == 0 and sample_clocks:
        sampler.start()
    kev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = sim.kernel_launches
    barrier()
    t0.record(stream)
    diag = None
    for i in range(steps):
        diag = hot_path(kev[i])
    t1.record(stream)
    barrier()
    clocks = sampler.stop() if (rank == 0 and sample_clocks) else None
    launches = sim.kernel_launches - l0
    ms_total = t0.elapsed_time(t1)
    ms_kernels = sum(a.elapsed_time(b) for a, b in kev)
    (ms_total, ms_kernels), (launches,) = reduce_over_ranks([ms_total, ms_kernels], [launches], world, "cuda")
    value = aggregate_value(S, SUBSTEPS, steps, world, ms_total)
    launch_ms = ms_kernels / (steps * main_launches)
    algorithmic = S * spl * bpu                                  # north_star: 16 B (32 B) per site-update, single-step roofline
    achieved = algorithmic / (launch_ms * 1e-3) / 1e9
    peak, peak_src = measured_peak_gbs()
    traffic, traffic_src = ncu_traffic_for(launch)
    compulsory = S * bpu                                         # one read + one write of both fields per LAUNCH (16/s B per site-update)
    own = {"compulsory_bytes_per_launch": compulsory,
           "frac_of_compulsory_traffic": compulsory / (launch_ms * 1e-3) / 1e9 / peak}
    if traffic:
        own["frac_of_own_traffic"] = traffic / (launch_ms * 1e-3) / 1e9 / peak
    else:
        own["frac_of_own_traffic"] = None
    kernel_name = {1: "generic", 2: "tiled", 3: "tb2", 4: "tbs", 5: "cluster"}.get(sim.get_info(binding.INFO_STEP_KERNEL), "?")
    fbytes = S * (4 if prec == 0 else 8)

    # ---- end to end through the C ABI with host buffers (pinned), copies inside the timed region
    e2e = None
    if with_e2e:
        try:
            dt = torch.float32 if prec == 0 else torch.float64
            hphi = torch.empty(S, dtype=dt, pin_memory=True)
            hpd = torch.empty(S, dtype=dt, pin_memory=True)
            sim.copy_out_to(hphi, hpd)
            n_e2e = max(1, min(steps, 2))
            step0 = sim.get_info(binding.INFO_STEP)

            def e2e_step(k):
                sim.copy_in(hphi, hpd, eta0=1.0, step=step0 + k * SUBSTEPS)
                sim.step(SUBSTEPS)
                d = sim.diagnostics()
                sim.copy_out_to(hphi, hpd)
                return d

            e2e_step(0)                                            # warm the copy path once
            barrier()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            for k in range(n_e2e):
                e2e_step(k + 1)
            b.record(stream)
            barrier()
            ms_e2e = a.elapsed_time(b)
            (ms_e2e,), _ = reduce_over_ranks([ms_e2e], [], world, "cuda")
            e2e = {"value": aggregate_value(S, SUBSTEPS, n_e2e, world, ms_e2e), "unit": UNIT,
                   "h2d_bytes_per_step": 2 * fbytes, "d2h_bytes_per_step": 2 * fbytes + 24,
                   "steps": n_e2e, "ms_per_step": ms_e2e / n_e2e,
                   "what": "prs_copy_in(pinned host) + %d prs_step + prs_diagnostics + prs_copy_out(pinned host)" % SUBSTEPS}
            del hphi, hpd
        except Exception as exc:                                   # e.g. not enough pinned host memory
            e2e = {"value": None, "unit": UNIT, "h2d_bytes_per_step": 2 * fbytes, "d2h_bytes_per_step": 2 * fbytes + 24,
                   "error": str(exc)[:200]}
    # ---- lattices that fit in L2 are bound by launches and host round trips, not by HBM: report the cycle at the
    # config's own cadence three ways -- one prs_step + prs_diagnostics call per cycle, prs_run (all cycles queued,
    # records read back once), and the step kernels alone
    small = None
    if 4 * fbytes <= (64 << 20):
        cad = OWN_CADENCE.get(config, SUBSTEPS)
        ncyc = max(20, 2000 // cad)

        def timed(fn):
            fn()
            barrier()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            fn()
            b.record(stream)
            barrier()
            return a.elapsed_time(b) * 1e3 / (ncyc * cad)           # us per PRS step

        def per_call():
            for _ in range(ncyc):
                sim.step(cad)
                sim.diagnostics()

        small = {"cycle": "%d PRS steps + 1 diagnostics pass, %d cycles" % (cad, ncyc),
                 "us_per_step_one_call_per_cycle": timed(per_call),
                 "us_per_step_prs_run": timed(lambda: sim.run(ncyc, cad)),
                 "us_per_step_step_kernels_only": timed(lambda: sim.step(ncyc * cad)),
                 "steps_per_s_prs_run": None,
                 "note": "state fits in L2: HBM fractions are meaningless here; the figures are launch- and latency-bound"}
        small["steps_per_s_prs_run"] = 1e6 / small["us_per_step_prs_run"]
        # One small box keeps 16 of the 148 SMs busy (small boxes under-use a GPU).  The paper's
        # answer is an ensemble -- five seeds per configuration (:119): independent handles on streams of their own, one
        # host thread each (prs_run blocks its caller), run side by side on the one GPU.
        try:
            small["ensemble_on_one_gpu"] = ensemble_leg(prs, torch, stream, dims, N, prec, era_m, ncyc, cad, S)
        except Exception as exc:
            small["ensemble_on_one_gpu"] = {"error": str(exc)[:200]}
    out = {
        "value": value, "unit": UNIT, "dtype": "f32" if prec == 0 else "f64", "steps": steps, "warmup": warmup,
        "ms_per_step": ms_total / steps, "gpu_launches": launches, "clocks": clocks, "e2e": e2e,
        "config": {"workload": config, "dims": dims, "N": N, "era_m": era_m, "alpha": 3.0, "deta": 0.1,
                   "W0": 10.0, "substeps_per_step": SUBSTEPS, "diagnostics_per_step": 1,
                   "parallelism": "replicas x%d (no sharding, no collective)" % world,
                   "l2": "state (%.1f GiB) exceeds L2; no flush needed" % (4 * fbytes / 2 ** 30) if 4 * fbytes > (1 << 28)
                         else "state (%.1f MiB) fits in L2: HBM fractions are not meaningful for this workload" % (4 * fbytes / 2 ** 20),
                   "step_kernel": kernel_name},
        "roofline": dict({"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                          "traffic": traffic, "traffic_source": traffic_src,
                          "what": "achieved / frac: the north_star single-step roofline (16 B FP32 / 32 B FP64 per site-update x "
                                  "site-updates per launch / launch time): above 1 because one launch advances several steps per "
                                  "pass over HBM; frac_of_own_traffic: measured DRAM bytes per launch / launch time / peak, i.e. "
                                  "how close the kernel is to being HBM-bound on the bytes it really moves",
                          "kernel": launch["kernel"], "grid": launch["grid"], "block": launch["block"],
                          "steps_per_launch": spl, "launches_timed": steps * main_launches, "launch_ms": launch_ms,
                          "peak_source": peak_src, "algorithmic_bytes_per_launch": algorithmic,
                          "step_kernel_share_of_step": ms_kernels / ms_total}, **own),
        "last_diag": {k: diag[k] for k in ("step", "eta", "link_count", "wall_sites", "rho", "gv2")},
        "small_lattice": small,
    }
    sim.close()
    del sim
    torch.cuda.empty_cache()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default=DEFAULT_CONFIG, choices=sorted(CONFIGS))
    ap.add_argument("--kernel", default=None, choices=["generic", "tiled", "tb2", "tbs"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--tbs-rows", type=int, default=0, choices=[0, 1, 2],
                    help="3D multi-step kernel: rows per thread (PRS_OPT_TBS_ROWS; 0 = the library's choice)")
    ap.add_argument("--tbs-loader", type=int, default=0, choices=[0, 1, 2],
                    help="3D multi-step kernel: ring loader (PRS_OPT_TBS_LOADER; 1 = cp.async, 0 / 2 = TMA bulk copies)")
    ap.add_argument("--no-also", action="store_true", help="skip the FP64 leg that follows the default workload")
    ap.add_argument("--decomposition", default="replicas", choices=["replicas", "slabs"],
                    help="replicas (default; the contract's line) or one lattice as z slabs (opt-in)")
    ap.add_argument("--slabs", type=int, default=8, help="single process, --decomposition slabs: slabs on this GPU")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
