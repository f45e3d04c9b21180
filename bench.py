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
DEFAULT_CONFIG = "3d_1024_f32_rad"
BYTES_PER_SITE_UPDATE = {0: 16, 1: 32}        # read phi, phidot; write phidot, phi

# dram__bytes_read.sum + dram__bytes_write.sum per step-kernel launch from the committed
# `ncu --set full` capture of the headline config (profiles/): filled in once measured.
NCU_TRAFFIC_BYTES_PER_LAUNCH = {
    # profiles/r01c_ncu_step3d_tbs4_f32_1024.md: 9.485 GB read + 8.558 GB written per four-step launch
    ("3d_1024_f32_rad", "tbs"): 18_043_506_000,
    # profiles/r01d_ncu_step3d_tbs4_f64_1024.md: 19.655 GB read + 17.151 GB written per four-step launch
    ("3d_1024_f64_rad", "tbs"): 36_806_144_000,
    # profiles/r01b_ncu_step3d_tb2_f32_1024.md: 9.136 GB read + 8.552 GB written per two-step launch
    ("3d_1024_f32_rad", "tb2"): 17_687_191_000,
    # profiles/r01b_ncu_step3d_tb2_f64_1024.md: 18.451 GB read + 17.144 GB written per two-step launch
    ("3d_1024_f64_rad", "tb2"): 35_594_988_000,
    # profiles/r01a_ncu_step3d_tiled_f32_1024.md: 8.867 GB read + 8.549 GB written per single-step launch
    ("3d_1024_f32_rad", "tiled"): 17_415_889_000,
    # profiles/r01e_ncu_step2d_tbs8_f32_16384.md: 2.572 GB read + 2.109 GB written per eight-step launch
    ("2d_16384_f32_rad", "tbs"): 4_680_775_000,
    # profiles/r01e_ncu_step2d_tbs6_f64_16384.md: 5.133 GB read + 4.260 GB written per six-step launch
    ("2d_16384_f64_rad", "tbs"): 9_392_606_000,
}


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


def oracle_sample(dims, prec, era_m, nsteps, threads, N=None, seed=1, with_init=True):
    """Times the oracle's step loop + one diagnostics pass on a bounded sample of the workload: same
    dimensionality, precision, parameters and seeded field, smaller box.  Returns
    (site_updates, seconds, description)."""
    from oracle import binding as ref

    if N is None:
        N = 512 if dims == 3 else 8192
    sim = ref.RefSim(dims, N, prec, era_m=era_m, seed=seed, threads=threads)
    sim.init(1.0)
    t0 = time.perf_counter()
    sim.step(nsteps)
    d = sim.diagnostics()
    dt = time.perf_counter() - t0
    sim.close()
    desc = "%dD %d^%d %s, %d PRS steps + 1 diagnostics pass, %d thread(s); rho=%.5f" % (
        dims, N, dims, "FP32" if prec == 0 else "FP64", nsteps, threads, d["rho"])
    return N ** dims * nsteps, dt, desc


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
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    dims, N, prec, era_m = CONFIGS[args.config]
    threads = host_threads()
    nsub = 10
    for _ in range(args.warmup if args.warmup < 2 else 1):       # one warm pass is enough for a CPU loop
        oracle_sample(dims, prec, era_m, 2, threads, N=256 if dims == 3 else 4096)
    total_updates, total_s, desc = 0, 0.0, ""
    for _ in range(args.steps):
        u, s, desc = oracle_sample(dims, prec, era_m, nsub, threads)
        total_updates += u
        total_s += s
    value = total_updates / total_s
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total_s / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if prec == 0 else "f64", "data": "synthetic",
        "config": {"workload": args.config, "dims": dims, "N": N, "era_m": era_m, "substeps": SUBSTEPS,
                   "note": "oracle timed on a bounded sample of this workload (see cpu_baseline.sample)"},
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
    sim = prs.Simulation(dims, N, prec, era_m=era_m, seed=rank + 1)
    if args.kernel:
        sim.set_step_kernel({"generic": prs.KERNEL_GENERIC, "tiled": prs.KERNEL_TILED, "tb2": prs.KERNEL_TB2,
                             "tbs": prs.KERNEL_TBS}[args.kernel])
    if args.tbs_rows != 1:
        sim.set_option(binding.OPT_TBS_ROWS, args.tbs_rows)
    sim.init(1.0)
    stream = torch.cuda.current_stream()

    def hot_path(ev=None):
        if ev:
            ev[0].record(stream)
        sim.step(SUBSTEPS)
        if ev:
            ev[1].record(stream)
        return sim.diagnostics()

    for _ in range(args.warmup):
        hot_path()
    # ---- timed region: exactly K steps, device clock, max over ranks
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    kev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = sim.kernel_launches
    barrier()
    t0.record(stream)
    diag = None
    for i in range(args.steps):
        diag = hot_path(kev[i])
    t1.record(stream)
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    launches = sim.kernel_launches - l0
    ms_total = t0.elapsed_time(t1)
    ms_kernels = sum(a.elapsed_time(b) for a, b in kev)
    (ms_total, ms_kernels), (launches,) = reduce_over_ranks([ms_total, ms_kernels], [launches], world, "cuda")
    value = aggregate_value(S, SUBSTEPS, args.steps, world, ms_total)
    step_kernel_launches = SUBSTEPS * args.steps
    step_kernel = sim.get_info(binding.INFO_STEP_KERNEL)
    # PRS steps the dominant kernel advances per launch; a prs_step(50) of the four-step kernel is 12
    # four-step launches and one two-step launch, so launch_ms is the time per steps_per_launch steps
    tbs_steps = 4 if dims == 3 else (8 if prec == 0 else 6)          # the library's defaults (prs.h, PRS_OPT_TBS_STEPS)
    steps_per_launch = {prs.KERNEL_TB2: 2, prs.KERNEL_TBS: tbs_steps}.get(step_kernel, 1)
    launch_ms = ms_kernels / (step_kernel_launches / steps_per_launch)
    achieved = S * steps_per_launch * bpu / (launch_ms * 1e-3) / 1e9
    peak, peak_src = measured_peak_gbs()
    kernel_name = {1: "generic", 2: "tiled", 3: "tb2", 4: "tbs"}.get(step_kernel, str(step_kernel))

    # ---- end to end through the C ABI with host buffers (pinned), copies inside the timed region
    e2e = None
    fbytes = S * (4 if prec == 0 else 8)
    try:
        dt = torch.float32 if prec == 0 else torch.float64
        hphi = torch.empty(S, dtype=dt, pin_memory=True)
        hpd = torch.empty(S, dtype=dt, pin_memory=True)
        sim.copy_out_to(hphi, hpd)
        n_e2e = max(1, min(args.steps, 2))
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

    # ---- oracle on the host cores, rank 0, N=1 only
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        threads = host_threads()
        u, s, desc = oracle_sample(dims, prec, era_m, 10, threads)
        u1, s1, desc1 = oracle_sample(dims, prec, era_m, 4, 1, N=256 if dims == 3 else 4096)
        cpu = {"value": u / s, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc,
               "single_thread_value": u1 / s1, "single_thread_sample": desc1}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32" if prec == 0 else "f64", "data": "synthetic",
            "config": {"workload": args.config, "dims": dims, "N": N, "era_m": era_m, "alpha": 3.0, "deta": 0.1,
                       "W0": 10.0, "substeps_per_step": SUBSTEPS, "diagnostics_per_step": 1,
                       "parallelism": "replicas x%d (no sharding, no collective)" % world,
                       "l2": "state (%.1f GiB) exceeds L2; no flush needed" % (4 * fbytes / 2 ** 30),
                       "step_kernel": kernel_name, "tbs_rows_per_thread": args.tbs_rows},
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": NCU_TRAFFIC_BYTES_PER_LAUNCH.get((args.config, kernel_name)),
                         "kernel": "step kernel", "launch_ms": launch_ms, "peak_source": peak_src,
                         "algorithmic_bytes_per_launch": S * steps_per_launch * bpu,
                         "step_kernel_share_of_step": ms_kernels / ms_total},
            "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
            "last_diag": {k: diag[k] for k in ("step", "eta", "link_count", "wall_sites", "rho", "gv2")},
        }
        print(json.dumps(line))
    sim.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default=DEFAULT_CONFIG, choices=sorted(CONFIGS))
    ap.add_argument("--kernel", default=None, choices=["generic", "tiled", "tb2", "tbs"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--tbs-rows", type=int, default=1, choices=[1, 2],
                    help="3D multi-step kernel: rows per thread (PRS_OPT_TBS_ROWS; 2 = step3d_tbr_kernel)")
    ap.add_argument("--decomposition", default="replicas", choices=["replicas", "slabs"],
                    help="replicas (default; the contract's line) or one lattice as z slabs (opt-in)")
    ap.add_argument("--slabs", type=int, default=8, help="single process, --decomposition slabs: slabs on this GPU")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
