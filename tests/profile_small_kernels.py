"""Drives the kernels that bench.py's default line does not dwell on, for ncu captures (profiles/r02c_*):

    python -m tests.profile_small_kernels diag      # 1024^3 FP32 on a formed network: sign_bits_kernel + bit_links_kernel,
                                                    # then prs_weighted_area on the same bits (bit_area_kernel)
    python -m tests.profile_small_kernels cluster   # 256^2 FP32, prs_run at cadence 10: step2d_cluster_kernel on 16 CTAs
    python -m tests.profile_small_kernels cluster1  # the same at cadence 1: a launch is 64 steps and 64 diagnostics passes
"""
import sys


def main():
    import paper_1710_10420_b200 as prs

    what = sys.argv[1] if len(sys.argv) > 1 else "diag"
    if what == "diag":
        sim = prs.Simulation(3, 1024, prs.F32, seed=1)
        sim.init(1.0)
        sim.step(1268)                                      # eta = 127.8: a few per cent of the sites touch a wall
        for _ in range(3):
            sim.step(4)
            d = sim.diagnostics()
            a, _ = sim.weighted_area()
        print("diag ok: step %d link_count %d wall_sites %d weighted area %.6e" % (d["step"], d["link_count"], d["wall_sites"], a))
    else:
        sim = prs.Simulation(2, 256, prs.F32, seed=1)
        sim.init(1.0)
        if what == "cluster1":
            sim.step(300)
            recs = sim.run(128, 1)
        else:
            recs = sim.run(127, 10)                         # BASELINE.json configs[0]: eta 1 -> 128, diagnostics every 10 steps
        print("cluster ok: %s, %d records, last link_count %d" % (sim.step_launch_info()["kernel"], len(recs), recs[-1]["link_count"]))
    sim.close()
    return 0


if __name__ == "__main__":
    sys.exit(main())
