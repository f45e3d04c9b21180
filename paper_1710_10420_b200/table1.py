#!/usr/bin/env python
"""The paper's validation workload (Table I) on this library: boxes of 2048^2
and 128^3, five fixed seeds, FP32 and FP64, scaling exponents mu (rho ~ eta^mu) and nu (gamma v ~
eta^nu) from a least-squares fit of the late part of each run (ln eta > 2.58), mean and standard error
over the seeds.

    python -m paper_1710_10420_b200.table1 [--seeds 5] [--every 10] [--json]

The paper never states its time step, wall thickness, initial conditions or run length, so this is the
same experiment with BASELINE.json's parameters (deta = 0.1, W0 = 10, uniform(-1,1) Philox initial
field, phidot = 0, radiation era, eta from 1 to N/2), not a reproduction of its digits: Table I is
context.  rho is reported with both estimators: the plain link count and Eq. 7's
orientation-weighted area (prs_weighted_area).  Everything runs through the C ABI on one GPU.
"""
import argparse
import json
import math

import numpy as np

from . import F32, F64, Simulation

FIT_FROM_LN_ETA = 2.58                      # PAPER.md:129, natural log (R12)


def run_one(dims, N, prec, seed, every):
    sim = Simulation(dims, N, prec, seed=seed)
    sim.init(1.0)
    nsamp = int(round((N / 2 - 1.0) / 0.1)) // every
    eta, rho, rho_w, gv = [], [], [], []
    for _ in range(nsamp):
        sim.step(every)
        d = sim.diagnostics()
        eta.append(d["eta"])
        rho.append(d["rho"])
        rho_w.append(sim.weighted_area()[1])
        gv.append(math.sqrt(d["gv2"]) if d["gv2"] > 0 else float("nan"))
    sim.close()
    eta, rho, rho_w, gv = map(np.array, (eta, rho, rho_w, gv))
    sel = np.log(eta) > FIT_FROM_LN_ETA

    def slope(y):
        ok = sel & np.isfinite(y) & (y > 0)
        return float(np.polyfit(np.log(eta[ok]), np.log(y[ok]), 1)[0])

    return {"mu": slope(rho), "mu_weighted": slope(rho_w), "nu": slope(gv)}


def mean_and_error(values):
    v = np.array(values)
    return float(v.mean()), float(v.std(ddof=1) / math.sqrt(len(v))) if len(v) > 1 else 0.0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--seeds", type=int, default=5)
    ap.add_argument("--every", type=int, default=10, help="diagnostics cadence in steps")
    ap.add_argument("--json", action="store_true")
    args = ap.parse_args()
    rows = []
    for dims, N in ((2, 2048), (3, 128)):
        for prec, name in ((F32, "FP32"), (F64, "FP64")):
            fits = [run_one(dims, N, prec, seed, args.every) for seed in range(1, args.seeds + 1)]
            row = {"box": "%d^%d" % (N, dims), "precision": name, "seeds": args.seeds}
            for key in ("mu", "mu_weighted", "nu"):
                row[key], row[key + "_err"] = mean_and_error([f[key] for f in fits])
            rows.append(row)
    if args.json:
        print(json.dumps(rows))
        return
    print("| box | precision | mu (link count) | mu (Eq. 7 weighted) | nu |")
    print("|---|---|---|---|---|")
    for r in rows:
        print("| %s | %s | %.4f +- %.4f | %.4f +- %.4f | %.4f +- %.4f |" % (
            r["box"], r["precision"], r["mu"], r["mu_err"], r["mu_weighted"], r["mu_weighted_err"], r["nu"], r["nu_err"]))


if __name__ == "__main__":
    main()
