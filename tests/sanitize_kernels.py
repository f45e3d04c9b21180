"""Drives every kernel of libprs on small ragged lattices: for runs under compute-sanitizer where that tool is
available, and -- since it is closed on this pool's GPUs -- with the library's race-hunting build:

    compute-sanitizer --tool racecheck|memcheck|initcheck|synccheck python -m tests.sanitize_kernels
    PRS_LIBRARY_VARIANT=jitter python -m tests.sanitize_kernels          # libprs_jitter.so: -DPRS_RACE_JITTER=1

The jitter build (csrc/prs_arith.cuh, build.py VARIANTS) puts random warp-uniform delays of up to 4 us before and after
every barrier, before every publication of a row to shared memory and inside the wall-site stack, so that an ordering
that holds only because the warps of a CTA run in step turns into a wrong bit here: every result is compared bit
for bit with the one-thread-per-site kernel, which has no shared memory and no barrier.

("Race detection / sanitizers".)  The default step kernels are shared-memory pipelines whose
correctness rests on one CTA barrier per plane and on cp.async group accounting; the sizes below make every
kind of tile appear: several tiles and z chunks, ragged last tiles in x and y, the periodic seam inside a tile,
lattices smaller than one tile.  Each result is also compared bit for bit with the generic one-thread-per-site
kernel, so a run is a (small) parity test as well.  The summaries of the last run are in profiles/.
"""
import os
import sys

import numpy as np


def main():
    import torch

    import paper_1710_10420_b200 as prs
    from paper_1710_10420_b200 import prs as binding
    from paper_1710_10420_b200 import sharded
    from tests import fieldgen as fg

    assert torch.cuda.is_available()
    NP = {prs.F32: np.float32, prs.F64: np.float64}
    launches = 0

    def run(dims, N, prec, kernel, nsteps, opts=(), chunk=0):
        nonlocal launches
        phi, pd = fg.random_state(dims, N, 5, NP[prec])
        g = prs.Simulation(dims, N, prec, era_m=2.0)
        g.set_step_kernel(kernel)
        for o, v in opts:
            g.set_option(o, v)
        if chunk:
            g.set_option(binding.OPT_CHUNK, chunk)
        g.copy_in(phi, pd, eta0=1.0, step=3)
        g.step(nsteps)
        out = g.copy_out()
        launches += g.kernel_launches
        g.close()
        return out[0].tobytes(), out[1].tobytes()

    for prec in (prs.F32, prs.F64):
        for dims, sizes in ((3, (36, 68, 132)), (2, (36, 260))):
            for N in sizes:
                want = run(dims, N, prec, prs.KERNEL_GENERIC, 9)
                cases = [("tiled", prs.KERNEL_TILED, (), 0), ("tb2", prs.KERNEL_TB2, (), 0),
                         ("tbs3", prs.KERNEL_TBS, ((binding.OPT_TBS_STEPS, 3),), 0),
                         ("tbs4", prs.KERNEL_TBS, ((binding.OPT_TBS_STEPS, 4),), 0),
                         ("tbs4 short chunks", prs.KERNEL_TBS, ((binding.OPT_TBS_STEPS, 4),), 5)]
                if dims == 2:
                    cases += [("tbs6", prs.KERNEL_TBS, ((binding.OPT_TBS_STEPS, 6),), 0),
                              ("tbs8", prs.KERNEL_TBS, ((binding.OPT_TBS_STEPS, 8),), 0)]
                else:
                    cases += [("tbr3", prs.KERNEL_TBS, ((binding.OPT_TBS_STEPS, 3), (binding.OPT_TBS_ROWS, 2)), 0),
                              ("tbr4", prs.KERNEL_TBS, ((binding.OPT_TBS_STEPS, 4), (binding.OPT_TBS_ROWS, 2)), 0)]
                for name, kernel, opts, chunk in cases:
                    got = run(dims, N, prec, kernel, 9, opts, chunk)
                    assert got == want, (name, dims, N, prec)
                    print("ok step %-18s %dD N=%-4d %s" % (name, dims, N, "f32" if prec == prs.F32 else "f64"), flush=True)
        for N in (64, 128, 256):                                  # cluster-resident small-box kernel (256: 16 CTAs)
            want = run(2, N, prec, prs.KERNEL_GENERIC, 35)
            assert run(2, N, prec, prs.KERNEL_CLUSTER, 35) == want
            # ... and with the diagnostics passes inside its launches (prs_run): counts against the generic kernels'
            a, b2 = prs.Simulation(2, N, prec, seed=4), prs.Simulation(2, N, prec, seed=4)
            a.set_step_kernel(prs.KERNEL_CLUSTER)
            b2.set_step_kernel(prs.KERNEL_GENERIC)
            b2.set_option(binding.OPT_DIAG_KERNEL, prs.KERNEL_GENERIC)
            a.init(1.0)
            b2.init(1.0)
            recs = a.run(23, 7)
            for rcd in recs:
                b2.step(7)
                d = b2.diagnostics()
                assert (rcd["link_count"], rcd["wall_sites"]) == (d["link_count"], d["wall_sites"]), (N, prec, rcd["step"])
                assert abs(rcd["sum_ratio"] - d["sum_ratio"]) <= 1e-10 * d["sum_ratio"]
            pa, pb = a.copy_out(), b2.copy_out()
            assert pa[0].tobytes() == pb[0].tobytes() and pa[1].tobytes() == pb[1].tobytes()
            launches += a.kernel_launches + b2.kernel_launches
            a.close()
            b2.close()
            print("ok step cluster            2D N=%-4d %s" % (N, "f32" if prec == prs.F32 else "f64"), flush=True)
        # diagnostics (tiled and generic) and the weighted area, early and on a forming network
        for dims, N in ((3, 68), (3, 132), (2, 260), (3, 128), (2, 256)):
            res = []
            W = 4 if prec == prs.F32 else 2
            for dk in (prs.KERNEL_GENERIC, prs.KERNEL_TILED) + ((prs.KERNEL_BITS,) if N % (32 * W) == 0 else ()):
                g = prs.Simulation(dims, N, prec, seed=4)
                g.set_option(binding.OPT_DIAG_KERNEL, dk)
                g.init(1.0)
                row = []
                for k in (0, 40, 160):
                    g.step(k)
                    d = g.diagnostics()
                    row.append((d["link_count"], d["wall_sites"], g.weighted_area()[0]))
                res.append(row)
                launches += g.kernel_launches
                g.close()
            assert all([(a, b) for a, b, _ in res[0]] == [(a, b) for a, b, _ in r] for r in res[1:])
            print("ok diagnostics + weighted area %dD N=%-4d %s" % (dims, N, "f32" if prec == prs.F32 else "f64"), flush=True)
        # a lattice as two and three z slabs (init_slab_kernel, plane-range launches, halo copies)
        for N, world in ((68, 2), (132, 3)):
            whole = prs.Simulation(3, N, prec, seed=11)
            group = sharded.SlabGroup(N, [0] * world, prec, seed=11)
            whole.init(1.0)
            group.init(1.0)
            for k in (4, 3, 2, 1, 8):
                whole.step(k)
                group.step(k)
            a, b = whole.copy_out(), group.copy_out()
            assert a[0].tobytes() == b[0].tobytes() and a[1].tobytes() == b[1].tobytes()
            dw, dg = whole.diagnostics(), group.diagnostics()
            assert dw["link_count"] == dg["link_count"] and dw["wall_sites"] == dg["wall_sites"]
            assert abs(group.weighted_area()[0] - whole.weighted_area()[0]) <= 1e-12 * whole.weighted_area()[0]
            launches += whole.kernel_launches + group.kernel_launches
            group.close()
            whole.close()
            print("ok slabs N=%d x%d %s" % (N, world, "f32" if prec == prs.F32 else "f64"), flush=True)
    from paper_1710_10420_b200 import build as prs_build

    print("sanitize_kernels: all kernels of %s ran, %d launches, results identical to the generic kernel"
          % (os.path.basename(prs_build.lib_path(os.environ.get("PRS_LIBRARY_VARIANT", ""))), launches))
    return 0


if __name__ == "__main__":
    sys.exit(main())
