"""GPU parity: libprs (through its C ABI) against the CPU oracle on the same seeded inputs.

Bars (BASELINE.json north_star): link count bit-exact on any snapshot; fields after 20 steps within
1e-12 (FP64) / 2e-5 (FP32) of the oracle as the paper prints the update (LITERAL arithmetic).  On top
of that, with the same arithmetic form on both sides (FMA, COEF or LITERAL; R13) the fields
must be IDENTICAL bit for bit: IEEE-754 fixes every operation of each form, and neither side ever
contracts (or splits) a multiply-add that the form does not prescribe.
"""
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import paper_1710_10420_b200 as prs  # noqa: E402
from oracle import binding as ref  # noqa: E402
from paper_1710_10420_b200 import prs as binding  # noqa: E402
from tests import fieldgen as fg  # noqa: E402

NP = {prs.F32: np.float32, prs.F64: np.float64}
TOL = {prs.F32: 2e-5, prs.F64: 1e-12}
THREADS = max(1, min(32, len(os.sched_getaffinity(0))))
KERNELS = [prs.KERNEL_GENERIC, prs.KERNEL_TILED, prs.KERNEL_TB2, prs.KERNEL_TBS]


def make_pair(dims, N, prec, arith_gpu=prs.ARITH_FMA, arith_ref=ref.ARITH_LITERAL, kernel=prs.KERNEL_AUTO, **kw):
    g = prs.Simulation(dims, N, prec, **kw)
    g.set_arith(arith_gpu)
    g.set_step_kernel(kernel)
    r = ref.RefSim(dims, N, prec, arith=arith_ref, threads=THREADS, **kw)
    return g, r


def maxdiff(a, b):
    return float(np.max(np.abs(a.astype(np.float64) - b.astype(np.float64))))


# ------------------------------------------------------------------ T1: initial condition

@pytest.mark.parametrize("dims,N", [(2, 1), (2, 5), (2, 256), (2, 1000), (3, 3), (3, 64), (3, 101)])
@pytest.mark.parametrize("prec", [prs.F32, prs.F64])
@pytest.mark.parametrize("seed", [0, 1, (1 << 32) + 7])
def test_init_is_byte_identical(dims, N, prec, seed):
    g, r = make_pair(dims, N, prec, seed=seed, phi0=1.0 if seed != 1 else 1.75)
    g.init(1.0)
    r.init(1.0)
    gp, gv = g.copy_out()
    rp, rv = r.copy_out()
    assert gp.tobytes() == rp.tobytes() and gv.tobytes() == rv.tobytes()
    assert not np.any(np.signbit(gv))


def test_init_reproduces_the_printed_field_values():
    """SURVEY.md Appendix B's printed field values (tests/golden/philox_field_values.txt) through prs_init +
    prs_copy_out: seeds 42 and 0 on a small lattice in both precisions, and the printed block on the 64-bit path
    (seed 2^32+7, q = 2^32+1, i.e. sites 4q..4q+3) through a z slab of a 4096^3 lattice whose first owned plane
    z = 1024 starts at site 2^34 (the only way to hold such a site index on one GPU)."""
    from paper_1710_10420_b200 import sharded
    from tests.goldenio import read_philox_field_values

    values, blocks = read_philox_field_values()
    for prec in (prs.F32, prs.F64):
        for seed in (42, 0):
            for dims, N in ((2, 8), (3, 4)):
                g = prs.Simulation(dims, N, prec, seed=seed)
                g.init(1.0)
                flat = g.copy_out()[0].ravel()
                g.close()
                for sd, site, _, phi in values:
                    if sd == seed:
                        assert float(flat[site]) == phi, (prec, seed, site)
    N, z_begin = 4096, 1024
    for seed, q, words in blocks:
        s0 = 4 * q
        assert z_begin * N * N <= s0 < (z_begin + 4) * N * N
        slab = sharded.SlabSimulation(N, z_begin, 4, prs.F32, seed=seed)
        slab.init(1.0)
        flat = slab.copy_out()[0].ravel()                      # owned planes: global sites z_begin*N*N ...
        slab.close()
        off = s0 - z_begin * N * N
        want = [(2 * (w >> 8) + 1 - (1 << 24)) / float(1 << 24) for w in words]
        assert [float(v) for v in flat[off:off + 4]] == want


# ------------------------------------------------------------------ T2: 20 steps from the seeded state

CASES_2D = [4, 36, 132, 256, 520]
CASES_3D = [4, 20, 36, 64, 132]


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("prec", [prs.F32, prs.F64])
@pytest.mark.parametrize("dims,N", [(2, n) for n in CASES_2D] + [(3, n) for n in CASES_3D])
@pytest.mark.parametrize("era_m", [1.0, 2.0])
def test_20_steps_match_the_oracle(kernel, prec, dims, N, era_m):
    # (a) tolerance bar against the paper's literal form, GPU in its default (FMA) form
    g, r = make_pair(dims, N, prec, kernel=kernel, era_m=era_m, seed=3)
    g.init(1.0)
    r.init(1.0)
    g.step(20)
    r.step(20)
    gp, gv = g.copy_out()
    rp, rv = r.copy_out()
    assert maxdiff(gp, rp) <= TOL[prec] and maxdiff(gv, rv) <= TOL[prec]
    assert g.get_info(binding.INFO_STEP_KERNEL) == kernel
    assert g.get_info(binding.INFO_STEP) == 20
    # (b) same arithmetic form on both sides -> identical bits
    for ag, ar in ((prs.ARITH_FMA, ref.ARITH_FMA), (prs.ARITH_COEF, ref.ARITH_COEF), (prs.ARITH_LITERAL, ref.ARITH_LITERAL)):
        g2, r2 = make_pair(dims, N, prec, arith_gpu=ag, arith_ref=ar, kernel=kernel, era_m=era_m, seed=3)
        g2.init(1.0)
        r2.init(1.0)
        g2.step(20)
        r2.step(20)
        a, b = g2.copy_out(), r2.copy_out()
        assert a[0].tobytes() == b[0].tobytes() and a[1].tobytes() == b[1].tobytes()


@pytest.mark.parametrize("prec", [prs.F32, prs.F64])
@pytest.mark.parametrize("dims,N", [(2, 7), (2, 130), (3, 5), (3, 33)])
def test_sizes_only_the_generic_kernel_takes(prec, dims, N):
    g, r = make_pair(dims, N, prec, arith_ref=ref.ARITH_FMA, seed=9)
    g.init(1.0)
    r.init(1.0)
    g.step(20)
    r.step(20)
    a, b = g.copy_out(), r.copy_out()
    assert a[0].tobytes() == b[0].tobytes() and a[1].tobytes() == b[1].tobytes()
    W = 4 if prec == prs.F32 else 2
    if N % W:
        assert g.get_info(binding.INFO_STEP_KERNEL) == prs.KERNEL_GENERIC
        with pytest.raises(prs.PrsError):
            g.set_step_kernel(prs.KERNEL_TILED)


@pytest.mark.parametrize("prec", [prs.F32, prs.F64])
@pytest.mark.parametrize("dims,N", [(2, 260), (3, 68)])
@pytest.mark.parametrize("chunk,tile_y,tb2_tile_y", [(1, 4, 4), (3, 8, 8), (7, 16, 12), (1000, 8, 12)])
def test_tiling_parameters_do_not_change_a_bit(prec, dims, N, chunk, tile_y, tb2_tile_y):
    phi, pd = fg.random_state(dims, N, 77, NP[prec])
    outs = []
    kernels = [(prs.KERNEL_GENERIC, 0), (prs.KERNEL_TILED, chunk), (prs.KERNEL_TB2, chunk)]
    kernels.append((prs.KERNEL_TBS, chunk))
    for kernel, ch in kernels:
        g = prs.Simulation(dims, N, prec)
        g.set_step_kernel(kernel)
        if kernel == prs.KERNEL_TBS:
            g.set_option(binding.OPT_TBS_STEPS, 3 if chunk % 2 else 4)
        g.set_option(binding.OPT_CHUNK, ch)
        g.set_option(binding.OPT_TILE_Y, tile_y)
        g.set_option(binding.OPT_TB2_TILE_Y, tb2_tile_y)
        g.copy_in(phi, pd, eta0=2.0, step=5)
        g.step(6)
        outs.append(g.copy_out())
    for o in outs[1:]:
        assert outs[0][0].tobytes() == o[0].tobytes() and outs[0][1].tobytes() == o[1].tobytes()


# ------------------------------------------------------------------ T6: temporal blocking == single steps

@pytest.mark.parametrize("prec", [prs.F32, prs.F64])
@pytest.mark.parametrize("dims,N", [(2, 4), (2, 8), (2, 120), (2, 124), (2, 1024), (3, 4), (3, 8), (3, 60), (3, 124), (3, 200)])
@pytest.mark.parametrize("nsteps", [1, 2, 7])
def test_two_step_kernel_equals_single_steps_bitwise(prec, dims, N, nsteps):
    phi, pd = fg.random_state(dims, N, 5, NP[prec])
    outs = []
    for kernel in (prs.KERNEL_TILED, prs.KERNEL_TB2):
        g = prs.Simulation(dims, N, prec, era_m=2.0)
        g.set_step_kernel(kernel)
        g.copy_in(phi, pd, eta0=1.0, step=3)
        g.step(nsteps)
        outs.append(g.copy_out())
        assert g.get_info(binding.INFO_STEP) == 3 + nsteps
        # launches: two steps per launch, plus one single step for an odd remainder
        want = nsteps if kernel == prs.KERNEL_TILED else nsteps // 2 + nsteps % 2
        assert g.kernel_launches == want
    assert outs[0][0].tobytes() == outs[1][0].tobytes() and outs[0][1].tobytes() == outs[1][1].tobytes()


@pytest.mark.parametrize("prec", [prs.F32, prs.F64])
@pytest.mark.parametrize("dims,N", [(3, 4), (3, 8), (3, 20), (3, 36), (3, 60), (3, 124), (3, 200),
                                    (2, 4), (2, 8), (2, 36), (2, 120), (2, 124), (2, 260), (2, 1024)])
@pytest.mark.parametrize("S", [3, 4, 6, 8])
def test_multi_step_kernel_equals_single_steps_bitwise(prec, dims, N, S):
    if S > 4 and dims == 3:
        pytest.skip("pipelines of 6 and 8 stages exist in 2D only")
    phi, pd = fg.random_state(dims, N, 5, NP[prec])
    for arith in (prs.ARITH_FMA, prs.ARITH_COEF, prs.ARITH_LITERAL):
        for nsteps in (S, 2 * S + 1, 2 * S + 2, 11, 2 * S + 7):
            outs = []
            for kernel in (prs.KERNEL_TILED, prs.KERNEL_TBS):
                g = prs.Simulation(dims, N, prec, era_m=2.0)
                g.set_step_kernel(kernel)
                g.set_arith(arith)
                g.set_option(binding.OPT_TBS_STEPS, S)
                g.copy_in(phi, pd, eta0=1.0, step=3)
                g.step(nsteps)
                outs.append(g.copy_out())
                assert g.get_info(binding.INFO_STEP) == 3 + nsteps
                if kernel == prs.KERNEL_TBS:     # S-step launches, then the remainder in as few launches as there are instances for
                    mains, rest = nsteps // S, nsteps % S
                    if dims == 2 and prec == prs.F32 and S == 8 and rest == 2 and mains >= 1:
                        extra = 1                                 # the last 8 + 2 become 6 + 4: the same number of launches
                    elif dims == 2 and prec == prs.F64 and S == 6 and rest == 2 and mains >= 1:
                        extra = 0                                 # the last 6 + 2 become one eight-step launch
                    elif dims == 3 and S == 4 and rest == 2 and mains >= 1:
                        extra = 1                                 # the last 4 + 2 become 3 + 3
                    else:
                        extra = {0: 0, 1: 1, 2: 1, 3: 1, 4: 1, 5: 2, 6: 1 if dims == 2 else 2, 7: 2}[rest]
                    assert g.kernel_launches == mains + extra, (nsteps, S)
            assert outs[0][0].tobytes() == outs[1][0].tobytes() and outs[0][1].tobytes() == outs[1][1].tobytes()
            if arith != prs.ARITH_FMA:
                break                             # the other forms: one length is enough


@pytest.mark.parametrize("prec", [prs.F32, prs.F64])
@pytest.mark.parametrize("N", [4, 8, 20, 36, 60, 124, 200])
@pytest.mark.parametrize("S", [3, 4])
def test_two_rows_per_thread_kernel_equals_single_steps_bitwise(prec, N, S):
    """PRS_OPT_TBS_ROWS = 2 (step3d_tbr_kernel): same stages, two adjacent rows of the tile per thread."""
    phi, pd = fg.random_state(3, N, 6, NP[prec])
    for arith in (prs.ARITH_FMA, prs.ARITH_COEF, prs.ARITH_LITERAL):
        for nsteps in (S, 2 * S + 1, 3 * S + 2):
            outs = []
            for kernel, rows in ((prs.KERNEL_TILED, 1), (prs.KERNEL_TBS, 2)):
                g = prs.Simulation(3, N, prec, era_m=1.0)
                g.set_step_kernel(kernel)
                g.set_arith(arith)
                g.set_option(binding.OPT_TBS_STEPS, S)
                g.set_option(binding.OPT_TBS_ROWS, rows)
                g.copy_in(phi, pd, eta0=1.0, step=2)
                g.step(nsteps)
                outs.append(g.copy_out())
                g.close()
            assert outs[0][0].tobytes() == outs[1][0].tobytes() and outs[0][1].tobytes() == outs[1][1].tobytes()
            if arith != prs.ARITH_FMA:
                break
    g = prs.Simulation(2, 64, prec)
    with pytest.raises(prs.PrsError):
        g.set_option(binding.OPT_TBS_ROWS, 2)                        # 3D only
    g.close()


@pytest.mark.parametrize("prec", [prs.F32, prs.F64])
@pytest.mark.parametrize("N", [64, 128, 256])
def test_cluster_resident_kernel_equals_single_steps_bitwise(prec, N):
    """Small-box kernel (state in the registers and shared memory of one cluster of 8 or 16 CTAs, the rows across a CTA
    boundary pushed into the neighbour's shared memory with st.async on mbarriers whose phase flips every second step):
    1 to 9, 31, 32, 33, 75 and 130 steps (launches of at most 64) against the single-step kernel, all arithmetic forms;
    and against the oracle."""
    phi, pd = fg.random_state(2, N, 5, NP[prec])
    for arith in (prs.ARITH_FMA, prs.ARITH_COEF, prs.ARITH_LITERAL):
        for nsteps in (1, 2, 3, 4, 5, 6, 7, 8, 9, 31, 32, 33, 75, 130) if arith == prs.ARITH_FMA else (33,):
            outs = []
            for kernel in (prs.KERNEL_TILED, prs.KERNEL_CLUSTER):
                g = prs.Simulation(2, N, prec, era_m=2.0)
                g.set_step_kernel(kernel)
                g.set_arith(arith)
                g.copy_in(phi, pd, eta0=1.0, step=3)
                g.step(nsteps)
                outs.append(g.copy_out())
                if kernel == prs.KERNEL_CLUSTER:
                    assert g.kernel_launches == (nsteps + 63) // 64
            assert outs[0][0].tobytes() == outs[1][0].tobytes() and outs[0][1].tobytes() == outs[1][1].tobytes()
    g = prs.Simulation(2, N, prec, seed=3)
    g.set_step_kernel(prs.KERNEL_CLUSTER)
    r = ref.RefSim(2, N, prec, seed=3, arith=ref.ARITH_FMA)
    g.init(1.0)
    r.init(1.0)
    g.step(40)
    r.step(40)
    a, b = g.copy_out(), r.copy_out()
    assert a[0].tobytes() == b[0].tobytes() and a[1].tobytes() == b[1].tobytes()
    with pytest.raises(prs.PrsError):
        prs.Simulation(2, 96, prec).set_step_kernel(prs.KERNEL_CLUSTER)
    with pytest.raises(prs.PrsError):
        prs.Simulation(3, 64, prec).set_step_kernel(prs.KERNEL_CLUSTER)


# ------------------------------------------------------------------ T3: diagnostics on snapshots

@pytest.mark.parametrize("diag_kernel", [prs.KERNEL_GENERIC, prs.KERNEL_TILED])
@pytest.mark.parametrize("prec", [prs.F32, prs.F64])
@pytest.mark.parametrize("dims,N", [(2, 1), (2, 2), (2, 4), (2, 5), (2, 256), (2, 520), (2, 1000), (3, 2), (3, 4), (3, 7),
                                    (3, 64), (3, 100), (3, 132)])
def test_diagnostics_match_on_snapshots(diag_kernel, prec, dims, N):
    g, r = make_pair(dims, N, prec, arith_ref=ref.ARITH_FMA, seed=4)
    W = 4 if prec == prs.F32 else 2
    if diag_kernel == prs.KERNEL_TILED and N % W:
        with pytest.raises(prs.PrsError):
            g.set_option(binding.OPT_DIAG_KERNEL, diag_kernel)
        return
    g.set_option(binding.OPT_DIAG_KERNEL, diag_kernel)
    g.init(1.0)
    r.init(1.0)
    for nsteps in (0, 20, 60):
        g.step(nsteps)
        r.step(nsteps)
        dg, dr = g.diagnostics(), r.diagnostics()
        gp, gv = g.copy_out()
        dsnap = ref.diagnostics_of(gp, gv)                       # oracle on the GPU's exact bytes
        for d in (dr, dsnap):
            assert dg["link_count"] == d["link_count"] and dg["wall_sites"] == d["wall_sites"]
            assert abs(dg["sum_ratio"] - d["sum_ratio"]) <= 1e-10 * max(d["sum_ratio"], 1e-300)
            assert abs(dg["gv2"] - d["gv2"]) <= 1e-10 * max(d["gv2"], 1e-300)
        assert dg["step"] == dr["step"] and dg["eta"] == dr["eta"] and dg["rho"] == dr["rho"]
        assert g.get_info(binding.INFO_DIAG_KERNEL) == diag_kernel


@pytest.mark.parametrize("prec", [prs.F32, prs.F64])
@pytest.mark.parametrize("dims,N", [(2, 128), (2, 256), (2, 1152), (3, 64), (3, 128), (3, 192), (3, 256)])
def test_sign_bit_diagnostics_match_on_snapshots(prec, dims, N):
    """PRS_KERNEL_BITS (prs_kernels_bits.cuh: a pass that packs one sign bit per site, a pass that counts links and
    wall sites on the bit words and fetches phidot at wall sites only) against the oracle on the GPU's exact bytes
    and against the one-pass tiled kernel: on the white-noise start (every site a wall site: the stack path at full
    load), while the network forms, and on a formed network (a few wall sites per warp)."""
    W = 4 if prec == prs.F32 else 2
    g = prs.Simulation(dims, N, prec, seed=4)
    if N % (32 * W):
        with pytest.raises(prs.PrsError) as e:
            g.set_option(binding.OPT_DIAG_KERNEL, prs.KERNEL_BITS)
        assert e.value.code == 2
        return
    g.init(1.0)
    for nsteps in (0, 20, 60, 300):
        g.step(nsteps)
        g.set_option(binding.OPT_DIAG_KERNEL, prs.KERNEL_BITS)
        db = g.diagnostics()
        assert g.get_info(binding.INFO_DIAG_KERNEL) == prs.KERNEL_BITS
        g.set_option(binding.OPT_DIAG_KERNEL, prs.KERNEL_TILED)
        dt = g.diagnostics()
        gp, gv = g.copy_out()
        do = ref.diagnostics_of(gp, gv)                          # oracle on the GPU's exact bytes
        for d in (dt, do):
            assert db["link_count"] == d["link_count"] and db["wall_sites"] == d["wall_sites"]
            assert abs(db["sum_ratio"] - d["sum_ratio"]) <= 1e-10 * max(d["sum_ratio"], 1e-300)
        assert db["rho"] == dt["rho"] and db["step"] == dt["step"] and db["eta"] == dt["eta"]
    # twice the same bits (the order of the double additions is fixed by the launch configuration)
    g.set_option(binding.OPT_DIAG_KERNEL, prs.KERNEL_BITS)
    assert g.diagnostics()["sum_ratio"] == g.diagnostics()["sum_ratio"]
    # special fields: the vacuum, a signed zero, a planar kink pair
    dt_np = NP[prec]
    vac = np.full((N,) * dims, -1.0, dt_np)
    g.copy_in(vac, np.zeros_like(vac))
    d = g.diagnostics()
    assert d["link_count"] == 0 and d["wall_sites"] == 0 and d["gv2"] == 0.0
    z = np.ones((N,) * dims, dt_np)
    z[(3,) * dims] = -0.0                                        # -0 is negative (sign bit), also at a group edge below
    z[(0,) * dims] = -0.5
    z[(N - 1,) * dims] = -0.25                                   # the periodic neighbour of site 0 in every direction
    g.copy_in(z, np.ones_like(z))
    d, do = g.diagnostics(), ref.diagnostics_of(z, np.ones_like(z))
    assert d["link_count"] == do["link_count"] and d["wall_sites"] == do["wall_sites"]
    assert abs(d["sum_ratio"] - do["sum_ratio"]) <= 1e-12 * do["sum_ratio"]
    phi = fg.kink_pair(dims, N, np.pi / 10.0, dtype=dt_np)
    g.copy_in(phi, np.zeros_like(phi))
    d = g.diagnostics()
    assert d["link_count"] == 2 * N ** (dims - 1) and d["wall_sites"] == 4 * N ** (dims - 1)
    g.close()


@pytest.mark.parametrize("prec", [prs.F32, prs.F64])
def test_diagnostics_of_special_fields(prec):
    dt = NP[prec]
    N = 64
    g = prs.Simulation(3, N, prec)
    # vacuum: nothing
    g.copy_in(np.full((N,) * 3, -1.0, dt), np.zeros((N,) * 3, dt))
    d = g.diagnostics()
    assert d["link_count"] == 0 and d["wall_sites"] == 0 and d["gv2"] == 0.0
    # planar kink pair: exact area
    phi = fg.kink_pair(3, N, np.pi / 10.0, dtype=dt)
    g.copy_in(phi, np.zeros_like(phi))
    d = g.diagnostics()
    assert d["link_count"] == 2 * N * N and d["wall_sites"] == 4 * N * N and d["rho"] == 2.0 / N
    # signed zeros: +0 positive, -0 negative
    z = np.ones((N,) * 3, dt)
    z[3, 4, 5] = -0.0
    g.copy_in(z, np.ones_like(z))
    d = g.diagnostics()
    assert d["link_count"] == 6 and d["wall_sites"] == 7
    dr = ref.diagnostics_of(z, np.ones_like(z))
    assert abs(d["sum_ratio"] - dr["sum_ratio"]) <= 1e-12 * dr["sum_ratio"]


# ------------------------------------------------------------------ Eq. 2 with beta != 0 (exact equations)

@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("prec", [prs.F32, prs.F64])
@pytest.mark.parametrize("dims,N", [(2, 132), (3, 36)])
def test_exact_equations_alpha_beta_two_match_the_oracle(kernel, prec, dims, N):
    g = prs.Simulation(dims, N, prec, alpha=2.0, era_m=2.0, seed=8)
    g.set_step_kernel(kernel)
    g.set_beta(2.0)
    r = ref.RefSim(dims, N, prec, alpha=2.0, era_m=2.0, seed=8, beta=2.0, arith=ref.ARITH_FMA, threads=THREADS)
    g.init(1.5)
    r.init(1.5)
    g.step(20)
    r.step(20)
    a, b = g.copy_out(), r.copy_out()
    assert a[0].tobytes() == b[0].tobytes() and a[1].tobytes() == b[1].tobytes()
    lit = ref.RefSim(dims, N, prec, alpha=2.0, era_m=2.0, seed=8, beta=2.0, threads=THREADS)
    lit.init(1.5)
    lit.step(20)
    c = lit.copy_out()
    assert maxdiff(a[0], c[0]) <= TOL[prec] and maxdiff(a[1], c[1]) <= TOL[prec]
    pr = ref.RefSim(dims, N, prec, alpha=2.0, era_m=2.0, seed=8, arith=ref.ARITH_FMA, threads=THREADS)   # beta = 0
    pr.init(1.5)
    pr.step(20)
    assert pr.copy_out()[0].tobytes() != a[0].tobytes()


# ------------------------------------------------------------------ Eq. 7 with the PRS orientation weight

@pytest.mark.parametrize("prec", [prs.F32, prs.F64])
@pytest.mark.parametrize("dims,N", [(2, 1), (2, 2), (2, 5), (2, 256), (2, 1000), (3, 2), (3, 7), (3, 64), (3, 100)])
def test_weighted_area_matches_the_oracle_on_snapshots(prec, dims, N):
    g = prs.Simulation(dims, N, prec, seed=4)
    g.init(1.0)
    for nsteps in (0, 20, 60):
        g.step(nsteps)
        area, rho_w = g.weighted_area()
        gp, _ = g.copy_out()
        want = ref.weighted_area_of(gp)                      # oracle on the GPU's exact bytes
        assert abs(area - want) <= 1e-12 * max(want, 1.0)
        assert rho_w == area / N ** dims
        C = g.diagnostics()["link_count"]
        assert C / np.sqrt(dims) - 1e-9 <= area <= C + 1e-9


@pytest.mark.parametrize("prec", [prs.F32, prs.F64])
@pytest.mark.parametrize("dims,N", [(2, 2048), (3, 256)])
def test_weighted_area_on_the_packed_sign_bits(prec, dims, N):
    """From 2^22 sites up prs_weighted_area finds the crossing links as the set bits of the XOR words of the packed sign
    bits (bit_area_kernel) instead of marching the lattice: against the oracle on the GPU's exact bytes and against the
    marching kernel (forced through PRS_OPT_DIAG_KERNEL = TILED), early and on a formed network; the bit array left by
    prs_diagnostics is reused (one launch instead of two) and a step invalidates it."""
    g = prs.Simulation(dims, N, prec, seed=4)
    g.init(1.0)
    for nsteps in (0, 40, 300):
        g.step(nsteps)
        g.set_option(binding.OPT_DIAG_KERNEL, prs.KERNEL_AUTO)
        l0 = g.kernel_launches
        a_bits, rho_bits = g.weighted_area()
        assert g.kernel_launches - l0 == 2                       # sign bits + links
        l0 = g.kernel_launches
        assert g.weighted_area() == (a_bits, rho_bits)           # same bits, and the bit array was reused
        assert g.kernel_launches - l0 == 1
        g.set_option(binding.OPT_DIAG_KERNEL, prs.KERNEL_TILED)
        a_old, _ = g.weighted_area()
        want = ref.weighted_area_of(g.copy_out()[0])
        assert abs(a_bits - want) <= 1e-12 * want and abs(a_old - want) <= 1e-12 * want
        assert rho_bits == a_bits / N ** dims
    # a state that prs_diagnostics has just found dense in crossing links (the white-noise start) goes through the
    # marching kernel (one launch, no sign bits), a formed network through the bits; same value either way
    h2 = prs.Simulation(dims, N, prec, seed=4)
    h2.init(1.0)
    a_unknown, _ = h2.weighted_area()                           # nothing known about the state: the bits
    d = h2.diagnostics()
    assert d["link_count"] > 0.25 * dims * N ** dims
    l0 = h2.kernel_launches
    a_dense, _ = h2.weighted_area()
    assert h2.kernel_launches - l0 == 1 and abs(a_dense - a_unknown) <= 1e-12 * a_unknown
    h2.close()
    # prs_diagnostics (sign-bit pass) leaves the bits behind; a step invalidates them
    g.set_option(binding.OPT_DIAG_KERNEL, prs.KERNEL_BITS)
    d = g.diagnostics()
    l0 = g.kernel_launches
    a1, _ = g.weighted_area()
    assert g.kernel_launches - l0 == 1 and d["link_count"] / np.sqrt(dims) <= a1 <= d["link_count"]
    g.step(1)
    l0 = g.kernel_launches
    a2, _ = g.weighted_area()
    assert g.kernel_launches - l0 == 2 and a2 != a1
    assert abs(a2 - ref.weighted_area_of(g.copy_out()[0])) <= 1e-12 * a2
    # copy_in invalidates them as well
    phi = fg.kink_pair(dims, N, np.pi / 10.0, dtype=NP[prec])
    g.copy_in(phi, np.zeros_like(phi))
    assert g.weighted_area()[0] == 2.0 * N ** (dims - 1)           # walls normal to x: weight exactly 1
    g.close()


def test_weighted_area_of_special_fields():
    N = 64
    g = prs.Simulation(3, N, prs.F64)
    phi = fg.kink_pair(3, N, np.pi / 10.0, dtype=np.float64)
    g.copy_in(phi, np.zeros_like(phi))
    assert g.weighted_area()[0] == 2.0 * N * N               # walls normal to x: weight exactly 1
    diag = fg.plane_wave(3, N, (1, 1, 1))
    g.copy_in(diag, np.zeros_like(diag))
    area, _ = g.weighted_area()
    assert abs(area / g.diagnostics()["link_count"] - 1.0 / np.sqrt(3.0)) < 5e-3
    vac = np.full((N,) * 3, 1.0)
    g.copy_in(vac, np.zeros_like(vac))
    assert g.weighted_area() == (0.0, 0.0)


@pytest.mark.parametrize("dims,N,nsteps,ratio", [(3, 256, 300, 2.0 / 3.0), (2, 2048, 400, np.pi / 4.0)])
def test_weight_turns_the_link_count_into_the_area_of_an_isotropic_network(dims, N, nsteps, ratio):
    # Counting links overestimates the area of an isotropically oriented wall by the mean of
    # |n_x| + |n_y| (+ |n_z|) over directions: 4/pi in 2D, 3/2 in 3D; the PRS weight of Eq. 7 removes
    # exactly that, so weighted / unweighted -> pi/4 and 2/3 once the network has formed.
    g = prs.Simulation(dims, N, prs.F32, seed=6)
    g.init(1.0)
    g.step(nsteps)
    area, _ = g.weighted_area()
    assert abs(area / g.diagnostics()["link_count"] - ratio) < 0.02


# ------------------------------------------------------------------ symmetries on the GPU (P2-P5 re-run)

@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("prec", [prs.F32, prs.F64])
@pytest.mark.parametrize("dims,N", [(2, 136), (3, 36)])
def test_gpu_symmetries_are_bit_exact(kernel, prec, dims, N):
    dt = NP[prec]
    phi, pd = fg.random_state(dims, N, 13, dt)

    def run(p, v):
        g = prs.Simulation(dims, N, prec, era_m=2.0)
        g.set_step_kernel(kernel)
        g.copy_in(p, v, eta0=1.0, step=0)
        g.step(5)
        return g.copy_out()

    p0, v0 = run(phi, pd)
    p1, v1 = run(-phi, -pd)
    assert np.array_equal(p0, -p1) and np.array_equal(v0, -v1)
    sh = (5, 3, 1)[:dims]
    p2, v2 = run(fg.roll_state(phi, sh), fg.roll_state(pd, sh))
    assert np.array_equal(fg.roll_state(p0, sh), p2) and np.array_equal(fg.roll_state(v0, sh), v2)
    for ax in range(dims):
        p3, v3 = run(fg.flip_axis(phi, ax), fg.flip_axis(pd, ax))
        assert np.array_equal(fg.flip_axis(p0, ax), p3) and np.array_equal(fg.flip_axis(v0, ax), v3)
    vac = np.full((N,) * dims, 1.0, dt)
    pv, vv = run(vac, np.zeros_like(vac))
    assert np.array_equal(pv, vac) and np.all(vv == 0)


# ------------------------------------------------------------------ T4: restart parity at late times

@pytest.mark.parametrize("dims,N,prec,adv", [(2, 512, prs.F32, 600), (3, 96, prs.F32, 200), (3, 64, prs.F64, 150)])
def test_restart_parity(dims, N, prec, adv):
    g = prs.Simulation(dims, N, prec, seed=5)
    g.init(1.0)
    g.step(adv)
    gp, gv = g.copy_out()
    r = ref.RefSim(dims, N, prec, arith=ref.ARITH_FMA, threads=THREADS)
    r.copy_in(gp, gv, eta0=1.0, step=adv)
    g.step(20)
    r.step(20)
    a, b = g.copy_out(), r.copy_out()
    assert a[0].tobytes() == b[0].tobytes() and a[1].tobytes() == b[1].tobytes()
    dg, dr = g.diagnostics(), r.diagnostics()
    assert dg["link_count"] == dr["link_count"] and dg["wall_sites"] == dr["wall_sites"]
    assert dg["eta"] == dr["eta"]
    # and within tolerance of the literal form
    r2 = ref.RefSim(dims, N, prec, arith=ref.ARITH_LITERAL, threads=THREADS)
    r2.copy_in(gp, gv, eta0=1.0, step=adv)
    r2.step(20)
    c = r2.copy_out()
    assert maxdiff(a[0], c[0]) <= TOL[prec] and maxdiff(a[1], c[1]) <= TOL[prec]


# ------------------------------------------------------------------ T5: long-run curve, config 0 (256^2)

def fit_mu(etas, rhos, eta_fit):
    sel = (etas >= eta_fit) & (rhos > 0)
    return float(np.polyfit(np.log(etas[sel]), np.log(rhos[sel]), 1)[0])


def test_config0_256sq_full_run_curve():
    # BASELINE.json configs[0]: 2D 256^2 FP32, radiation era, eta 1 -> 128, link count every 10 steps;
    # the FP64 oracle is run as well.
    N, nsamp = 256, 127
    g = prs.Simulation(2, N, prs.F32, seed=1)
    r32 = ref.RefSim(2, N, ref.F32, seed=1, threads=THREADS)           # literal, FP32
    r64 = ref.RefSim(2, N, ref.F64, seed=1, threads=THREADS)           # literal, FP64
    for s in (g, r32, r64):
        s.init(1.0)
    eta, cg, c32, c64 = [], [], [], []
    for _ in range(nsamp):
        for s in (g, r32, r64):
            s.step(10)
        dg, d32, d64 = g.diagnostics(), r32.diagnostics(), r64.diagnostics()
        eta.append(dg["eta"]); cg.append(dg["rho"]); c32.append(d32["rho"]); c64.append(d64["rho"])
        assert dg["eta"] == d32["eta"]
    eta, cg, c32, c64 = map(np.array, (eta, cg, c32, c64))
    assert np.max(np.abs(cg - c32) / c32) <= 0.02
    assert np.max(np.abs(cg - c64) / c64) <= 0.02
    mu_g, mu_32, mu_64 = (fit_mu(eta, c, 13.2) for c in (cg, c32, c64))
    assert abs(mu_g - mu_32) <= 0.02 and abs(mu_g - mu_64) <= 0.02


@pytest.mark.parametrize("dims,N,era_m,every,nsamp", [
    (2, 1024, 2.0, 10, 127),      # 2D, matter era, eta 1 -> 128
    (3, 128, 1.0, 10, 63),        # 3D, radiation era, eta 1 -> 64 (the paper's own 3D box size)
    (3, 128, 2.0, 10, 63),        # 3D, matter era
])
def test_long_run_curves_match_the_oracle(dims, N, era_m, every, nsamp):
    """T5 at sizes the oracle runs in seconds: the whole run (default kernels and arithmetic) against
    the oracle's literal FP32 form: rho(eta) within 2 % at every sample, fitted exponent within 0.02."""
    g = prs.Simulation(dims, N, prs.F32, era_m=era_m, seed=3)
    r = ref.RefSim(dims, N, ref.F32, era_m=era_m, seed=3, threads=THREADS)
    g.init(1.0)
    r.init(1.0)
    eta, cg, cr = [], [], []
    for _ in range(nsamp):
        g.step(every)
        r.step(every)
        dg, dr = g.diagnostics(), r.diagnostics()
        assert dg["eta"] == dr["eta"] and dg["step"] == dr["step"]
        eta.append(dg["eta"]); cg.append(dg["rho"]); cr.append(dr["rho"])
    eta, cg, cr = map(np.array, (eta, cg, cr))
    assert np.max(np.abs(cg - cr) / cr) <= 0.02
    assert abs(fit_mu(eta, cg, 13.2) - fit_mu(eta, cr, 13.2)) <= 0.02
    assert g.get_info(binding.INFO_STEP_KERNEL) == prs.KERNEL_TBS


@pytest.mark.parametrize("dims,N,prec", [(3, 200, prs.F32), (3, 72, prs.F64), (2, 1500, prs.F32)])
def test_repeated_runs_are_identical(dims, N, prec):
    """The pipelined kernels exchange rows through shared memory under one barrier per iteration; a
    missing ordering would show up as run-to-run differences.  Five runs of the default path (several
    chunks, ragged tiles) must agree byte for byte, diagnostics' floating-point sum included."""
    outs = []
    for _ in range(5):
        g = prs.Simulation(dims, N, prec, seed=12)
        g.init(1.0)
        g.step(26)
        d = g.diagnostics()
        p, v = g.copy_out()
        outs.append((p.tobytes(), v.tobytes(), d["link_count"], d["wall_sites"], d["sum_ratio"], g.weighted_area()[0]))
        g.close()
    assert all(o == outs[0] for o in outs[1:])


@pytest.mark.slow
def test_largest_lattice_that_fits_2048_cubed():
    """Maximum size: 2048^3 FP32 = 8.6e9 sites, 137 GB of workspace, link counts beyond 2^32 and byte
    offsets beyond 2^35.  The oracle cannot hold it, so the default path (four-step kernel with unsigned
    32-bit vector cursors at their limit, tiled diagnostics) is checked against the generic kernels,
    whose index arithmetic is plain 64-bit: diagnostics equal, and the last 64 MiB of phi identical."""
    import ctypes
    import torch

    free, _ = torch.cuda.mem_get_info()
    need = prs.prs_workspace_bytes(3, 2048, prs.F32)
    if free < need + (1 << 30):
        pytest.skip("needs %.0f GB of free device memory" % (need / 1e9))
    cudart = ctypes.CDLL("libcudart.so")
    res = []
    for kernel in (prs.KERNEL_AUTO, prs.KERNEL_GENERIC):
        g = prs.Simulation(3, 2048, prs.F32, seed=2)
        g.set_step_kernel(kernel)
        if kernel == prs.KERNEL_GENERIC:
            g.set_option(binding.OPT_DIAG_KERNEL, prs.KERNEL_GENERIC)
        g.init(1.0)
        g.step(9)                                            # two four-step launches and a single step
        d = g.diagnostics()
        assert g.get_info(binding.INFO_STEP_KERNEL) == (prs.KERNEL_TBS if kernel == prs.KERNEL_AUTO else kernel)
        pp, _ = g.device_pointers()
        tail = torch.empty(1 << 24, dtype=torch.float32, device="cuda")
        off = (2048 ** 3 - (1 << 24)) * 4
        rc = cudart.cudaMemcpy(ctypes.c_void_p(tail.data_ptr()), ctypes.c_void_p(pp + off), ctypes.c_size_t((1 << 24) * 4), 3)
        assert rc == 0
        res.append((d["link_count"], d["wall_sites"], d["sum_ratio"], tail.cpu().numpy().tobytes()))
        g.close()
        del g, tail
        torch.cuda.empty_cache()
    assert res[0][0] == res[1][0] > 2 ** 32 and res[0][1] == res[1][1]
    assert abs(res[0][2] - res[1][2]) <= 1e-10 * res[1][2]
    assert res[0][3] == res[1][3]


@pytest.mark.slow
@pytest.mark.skipif(os.environ.get("PRS_LONG_RUNS") != "1",
                    reason="full-length oracle runs take ~15 min each on 16 cores; set PRS_LONG_RUNS=1")
@pytest.mark.parametrize("dims,N,era_m,every", [(2, 4096, 1.0, 100), (2, 4096, 2.0, 100), (3, 512, 1.0, 50)])
def test_full_length_runs_match_the_oracle(dims, N, era_m, every):
    """T5 at BASELINE.json's configs[1] and configs[3] in full: eta from 1 to N/2, diagnostics at the
    configs' cadence, the GPU's default path against the oracle's literal FP32 form on the host cores.
    rho(eta) within 2 % at every sample, fitted exponent within 0.02 (fit for eta >= 32); the last
    measured outcome is recorded in DESIGN.md section 10."""
    nsamp = int(round((N / 2 - 1.0) / 0.1)) // every
    g = prs.Simulation(dims, N, prs.F32, era_m=era_m, seed=1)
    r = ref.RefSim(dims, N, ref.F32, era_m=era_m, seed=1, threads=THREADS)
    g.init(1.0)
    r.init(1.0)
    eta, cg, cr, worst = [], [], [], 0.0
    for _ in range(nsamp):
        g.step(every)
        r.step(every)
        dg, dr = g.diagnostics(), r.diagnostics()
        assert dg["eta"] == dr["eta"]
        eta.append(dg["eta"]); cg.append(dg["rho"]); cr.append(dr["rho"])
        worst = max(worst, abs(dg["rho"] - dr["rho"]) / dr["rho"])
    eta, cg, cr = map(np.array, (eta, cg, cr))
    mu_g, mu_r = fit_mu(eta, cg, 32.0), fit_mu(eta, cr, 32.0)
    print("LONGRUN dims=%d N=%d era_m=%g samples=%d worst_rel_rho=%.3e mu_gpu=%.5f mu_oracle=%.5f identical_samples=%d"
          % (dims, N, era_m, nsamp, worst, mu_g, mu_r, int(np.sum(cg == cr))))
    assert worst <= 0.02 and abs(mu_g - mu_r) <= 0.02


def test_driver_smoke_entry_point_passes():
    """__graft_entry__.smoke() is what the driver runs on the GPU box before the bench: all four step
    kernels against the oracle on three small lattices."""
    import __graft_entry__ as entry

    entry.smoke()


# ------------------------------------------------------------------ state handling

def test_copy_in_out_roundtrip_device_and_host_and_step_split():
    import torch
    N = 128
    phi, pd = fg.random_state(2, N, 3, np.float32)
    g = prs.Simulation(2, N, prs.F32)
    tp, tv = torch.from_numpy(phi).cuda(), torch.from_numpy(pd).cuda()
    g.copy_in(tp, tv, eta0=1.5, step=2)                    # device pointers
    op, ov = torch.empty_like(tp), torch.empty_like(tv)
    g.copy_out_to(op, ov)
    assert torch.equal(op, tp) and torch.equal(ov, tv)
    g.step(3); g.step(0); g.step(4)
    a = g.copy_out()
    g2 = prs.Simulation(2, N, prs.F32)
    g2.copy_in(phi, pd, eta0=1.5, step=2)                  # host pointers
    g2.step(7)
    b = g2.copy_out()
    assert a[0].tobytes() == b[0].tobytes() and a[1].tobytes() == b[1].tobytes()
    assert g.get_info(binding.INFO_STEP) == 9 and g.diagnostics()["eta"] == 1.5 + 9 * 0.1
    # device_pointers view equals copy_out
    pp, pv = g.device_pointers()
    assert pp and pv and pp != pv
    assert g.kernel_launches >= 2              # 128^2: the cluster-resident kernel, one launch per prs_step call


def test_error_paths_on_device():
    g = prs.Simulation(2, 16, prs.F32)
    with pytest.raises(prs.PrsError) as e:
        g.step(1)
    assert e.value.code == 4
    with pytest.raises(prs.PrsError):
        g.diagnostics()
    with pytest.raises(prs.PrsError):
        g.init(-1.0)
    g.init(1.0)
    with pytest.raises(prs.PrsError):
        g.step(-1)
    with pytest.raises(prs.PrsError):
        g.set_option(99, 0)
    with pytest.raises(prs.PrsError):
        g.set_option(binding.OPT_TILE_Y, 5)


# ------------------------------------------------------------------ full sizes of BASELINE.json, bench.py's launch configuration

def chunked_maxdiff(a, b, chunk=1 << 26):
    fa, fb = a.reshape(-1), b.reshape(-1)
    m = 0.0
    for i in range(0, fa.size, chunk):
        m = max(m, float(np.max(np.abs(fa[i:i + chunk].astype(np.float64) - fb[i:i + chunk].astype(np.float64)))))
    return m


FULL_SIZE_CASES = [
    # dims, N, precision, era_m, literal too?   (configs[1] .. configs[4] of BASELINE.json; both eras and both
    # precisions appear at the headline size; the other era of each precision at 1024^3 starts from a formed
    # network in LATE_CASES below).  The north_star tolerance against the paper's LITERAL form is asserted at
    # one case per size and precision; bit-identity with the oracle's FMA form at every case.
    (2, 4096, prs.F32, 1.0, True), (2, 4096, prs.F32, 2.0, False),
    (2, 16384, prs.F32, 1.0, True), (2, 16384, prs.F64, 1.0, True),
    (3, 512, prs.F32, 1.0, True),
    (3, 1024, prs.F32, 1.0, False), (3, 1024, prs.F64, 2.0, False),      # LITERAL at 1024^3: LATE_CASES, "boxes+lit"
]


@pytest.mark.slow
@pytest.mark.parametrize("dims,N,prec,era_m,literal", FULL_SIZE_CASES)
def test_full_size_20_steps_match_the_oracle_everywhere(dims, N, prec, era_m, literal):
    """T2 at full size: default options (the kernel selection and tiling bench.py times), seeded
    initial state, 20 steps, every site compared with the oracle run on the host cores: identical
    bits against the oracle in the same arithmetic form, within the north_star tolerance against the
    paper's literal form (checked on phidot and phi), and the diagnostics of the final state."""
    g = prs.Simulation(dims, N, prec, era_m=era_m, seed=2)
    g.init(1.0)
    g.step(20)
    assert g.get_info(binding.INFO_STEP_KERNEL) == prs.KERNEL_TBS
    dg = g.diagnostics()
    gp, gv = g.copy_out()
    g.close()
    r = ref.RefSim(dims, N, prec, era_m=era_m, seed=2, arith=ref.ARITH_FMA, threads=THREADS)
    r.init(1.0)
    r.step(20)
    dr = r.diagnostics()
    rp, rv = r.copy_out()
    r.close()
    assert np.array_equal(gp, rp) and np.array_equal(gv, rv)
    assert dg["link_count"] == dr["link_count"] and dg["wall_sites"] == dr["wall_sites"]
    assert abs(dg["sum_ratio"] - dr["sum_ratio"]) <= 1e-10 * dr["sum_ratio"]
    del rp, rv
    if not literal:
        return
    r = ref.RefSim(dims, N, prec, era_m=era_m, seed=2, arith=ref.ARITH_LITERAL, threads=THREADS)
    r.init(1.0)
    r.step(20)
    lp, lv = r.copy_out()
    r.close()
    assert chunked_maxdiff(gp, lp) <= TOL[prec] and chunked_maxdiff(gv, lv) <= TOL[prec]


# ------------------------------------------------------------------ T3/T4 at full size on a FORMED network

def steps_to(eta):
    return int(round((eta - 1.0) / 0.1))


def wrapped_box(a, origin, M):
    """The M^d sub-lattice of the periodic array a whose corner is at `origin` (given in array-axis order)."""
    idx = [(o + np.arange(M)) % n for o, n in zip(origin, a.shape)]
    return np.ascontiguousarray(a[np.ix_(*idx)])


LATE_CASES = [
    # dims, N, precision, era_m, eta of the checkpoint, mode
    #   "all":   the oracle advances the WHOLE lattice 20 steps from the GPU's snapshot: every site compared
    #   "boxes": the oracle advances sub-lattices of the snapshot (sampled outputs: after k steps a site depends on
    #            the sites within k links of it, so the inner (M-40)^d sites of a periodic M^d copy of a box see
    #            exactly what they see in the whole lattice); boxes straddle the periodic seam, CTA tiles and z chunks
    #   "+lit":  also the north_star tolerance against the oracle's LITERAL form
    # Diagnostics and the weighted area of the checkpoint are compared on the whole lattice in every case.
    (2, 4096, prs.F32, 1.0, 512.0, "all+lit"), (2, 4096, prs.F32, 2.0, 1843.0, "all"),
    (2, 16384, prs.F32, 1.0, 7372.0, "all+lit"), (2, 16384, prs.F64, 1.0, 2048.0, "all+lit"),
    (3, 512, prs.F32, 1.0, 230.0, "all+lit"),
    (3, 1024, prs.F32, 2.0, 460.0, "all"), (3, 1024, prs.F64, 1.0, 128.0, "all"),
    (3, 1024, prs.F32, 1.0, 128.0, "boxes+lit"), (3, 1024, prs.F64, 2.0, 460.0, "boxes+lit"),
]


@pytest.mark.slow
@pytest.mark.parametrize("dims,N,prec,era_m,eta,mode", LATE_CASES)
def test_full_size_restart_parity_on_a_formed_network(dims, N, prec, era_m, eta, mode):
    """SURVEY 8(c) T3/T4 at BASELINE.json's full sizes, every precision and era (the paper's own
    validation compares sequential and parallel codes at LATE timesteps).  The GPU runs its default path to a
    checkpoint where the wall network has formed (eta = N/8 or 0.45 N: a few per cent of the sites touch a wall,
    which is where the diagnostics kernel's per-warp compaction and prs_weighted_area's link stack take their
    data-dependent paths), then: snapshot -> oracle; diagnostics and Eq. 7's weighted area of that snapshot
    against the oracle on the same bytes; 20 more steps on both sides; fields identical bit for bit against the
    oracle's FMA form (and within the north_star bar of its LITERAL form), diagnostics again."""
    adv = steps_to(eta)
    g = prs.Simulation(dims, N, prec, era_m=era_m, seed=1)
    g.init(1.0)
    g.step(adv)
    assert g.get_info(binding.INFO_STEP_KERNEL) == prs.KERNEL_TBS
    d0 = g.diagnostics()
    area0, _ = g.weighted_area()
    sp, sv = g.copy_out()                                       # the checkpoint
    o0 = ref.diagnostics_of(sp, sv)
    assert d0["link_count"] == o0["link_count"] and d0["wall_sites"] == o0["wall_sites"]
    assert abs(d0["sum_ratio"] - o0["sum_ratio"]) <= 1e-10 * o0["sum_ratio"]
    assert 0 < d0["wall_sites"] < 0.25 * N ** dims              # a formed network, not the white-noise start
    want = ref.weighted_area_of(sp)
    assert abs(area0 - want) <= 1e-12 * want
    assert d0["link_count"] / np.sqrt(dims) <= area0 <= d0["link_count"]
    g.step(20)
    d1 = g.diagnostics()
    if mode.startswith("all"):
        forms = [ref.ARITH_FMA] + ([ref.ARITH_LITERAL] if mode.endswith("+lit") else [])
        for arith in forms:
            r = ref.RefSim(dims, N, prec, era_m=era_m, arith=arith, threads=THREADS)
            r.copy_in(sp, sv, eta0=1.0, step=adv)
            if arith == forms[-1]:
                del sp, sv                                      # 1024^3 FP64: keep the host footprint down
            r.step(20)
            o1 = r.diagnostics()
            rp, rv = r.copy_out()
            r.close()
            gp, gv = g.copy_out()
            if arith == ref.ARITH_FMA:
                assert np.array_equal(gp, rp) and np.array_equal(gv, rv)
                assert d1["link_count"] == o1["link_count"] and d1["wall_sites"] == o1["wall_sites"]
                assert abs(d1["sum_ratio"] - o1["sum_ratio"]) <= 1e-10 * o1["sum_ratio"]
                assert d1["eta"] == o1["eta"] and d1["step"] == o1["step"] == adv + 20
            else:
                assert chunked_maxdiff(gp, rp) <= TOL[prec] and chunked_maxdiff(gv, rv) <= TOL[prec]
            del rp, rv, gp, gv
    else:
        M, R = 192, 20
        gp, gv = g.copy_out()
        assert d1["step"] == adv + 20 and 0 < d1["link_count"] < d0["link_count"]       # the network keeps thinning out
        # corners (z, y, x): the periodic seam in all axes; the seam of the z chunks of 128 planes and of the
        # 16-/20-row y tiles in mid-lattice; the x tiles (120 / 56 sites wide); one more in the bulk
        for origin in ((N - 70, N - 90, N - 100), (128 - 96, 512 - 100, 300), (640 - 50, 37, N - 130), (300, 700, 450)):
            bp, bv = wrapped_box(sp, origin, M), wrapped_box(sv, origin, M)
            ap, av = wrapped_box(gp, origin, M), wrapped_box(gv, origin, M)
            inner = (slice(R, M - R),) * dims
            for arith in [ref.ARITH_FMA] + ([ref.ARITH_LITERAL] if mode.endswith("+lit") else []):
                r = ref.RefSim(dims, M, prec, era_m=era_m, arith=arith, threads=THREADS)
                r.copy_in(bp, bv, eta0=1.0, step=adv)
                r.step(20)
                rp, rv = r.copy_out()
                r.close()
                if arith == ref.ARITH_FMA:
                    assert np.array_equal(ap[inner], rp[inner]) and np.array_equal(av[inner], rv[inner]), origin
                else:
                    assert maxdiff(ap[inner], rp[inner]) <= TOL[prec] and maxdiff(av[inner], rv[inner]) <= TOL[prec]
    g.close()


def test_race_hunting_build_gives_the_same_bits():
    """compute-sanitizer is closed on this pool's GPUs, so races are hunted with a second build of the same sources
    (-DPRS_RACE_JITTER=1: random warp-uniform delays of up to 4 us around every barrier, publication and stack push).
    tests/sanitize_kernels.py drives every kernel with it on ragged lattices and compares each result bit for bit with
    the generic kernel; an ordering that holds only because the warps run in step would fail there."""
    import subprocess
    import sys

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, PRS_LIBRARY_VARIANT="jitter")
    out = subprocess.run([sys.executable, "-m", "tests.sanitize_kernels"], cwd=root, env=env, stdout=subprocess.PIPE,
                         stderr=subprocess.STDOUT, text=True, timeout=900)
    assert out.returncode == 0, out.stdout[-3000:]
    assert "results identical to the generic kernel" in out.stdout
    assert "libprs_jitter.so" in out.stdout


@pytest.mark.parametrize("dims,N,prec,every,ncyc", [(2, 256, prs.F32, 10, 127), (2, 64, prs.F64, 1, 4100), (3, 64, prs.F32, 7, 9),
                                                   (3, 128, prs.F64, 50, 3), (2, 1000, prs.F32, 3, 5)])
def test_batched_cycles_equal_the_step_and_diagnostics_loop(dims, N, prec, every, ncyc):
    """prs_run(ncycles, steps_per_cycle) = the loop every BASELINE.json config runs, queued without a host round trip
    per cycle: every record must equal what prs_step + prs_diagnostics return, bit for bit (same kernels, same launch
    configuration), across the 4096-record ring on the device as well; the state afterwards is the same."""
    a = prs.Simulation(dims, N, prec, seed=3)
    b = prs.Simulation(dims, N, prec, seed=3)
    a.init(1.0)
    b.init(1.0)
    fused = dims == 2 and N in (64, 128, 256)                    # AUTO runs these cycles inside cluster-resident launches
    got = a.run(ncyc, every)
    assert len(got) == ncyc
    assert (a.get_info(binding.INFO_STEP_KERNEL) == prs.KERNEL_CLUSTER) == fused
    for i in range(ncyc):
        b.step(every)
        want = b.diagnostics()
        if i < 40 or i % 97 == 0 or i >= ncyc - 5:
            if fused:                                           # the cluster kernel measures inside its launches: the
                for k in ("step", "eta", "link_count", "wall_sites", "rho"):     # double sum is added in another order
                    assert got[i][k] == want[k], (i, k)
                assert abs(got[i]["sum_ratio"] - want["sum_ratio"]) <= 1e-10 * max(want["sum_ratio"], 1e-300)
                assert abs(got[i]["gv2"] - want["gv2"]) <= 1e-10 * max(want["gv2"], 1e-300)
            else:
                assert got[i] == want, i
    assert got[-1]["step"] == ncyc * every and a.get_info(binding.INFO_STEP) == ncyc * every
    pa, pb = a.copy_out(), b.copy_out()
    assert pa[0].tobytes() == pb[0].tobytes() and pa[1].tobytes() == pb[1].tobytes()
    assert a.run(0, 5) == [] and a.get_info(binding.INFO_STEP) == ncyc * every
    zero = a.run(2, 0)                                          # no steps: the same state measured twice
    assert zero[0] == zero[1] and zero[0]["step"] == ncyc * every
    a.close()
    b.close()


@pytest.mark.parametrize("dims,N,prec", [(2, 256, prs.F32), (2, 128, prs.F64), (2, 1024, prs.F32), (3, 64, prs.F32)])
def test_handles_on_streams_and_threads_of_their_own_run_side_by_side(dims, N, prec):
    """An ensemble of independent boxes on one GPU (PAPER.md:119: five seeds per configuration; :97, :111: a small box
    under-uses the GPU): six handles, each on a stream of its own, each driven by its own host thread through prs_run,
    all at once -- records and fields equal to the same seeds run one after the other on the default stream.  (Exercises
    the library's process-wide state -- per-device kernel attributes, the 16-CTA cluster probe -- under concurrent calls,
    and clusters of different handles resident on the GPU together.)"""
    import threading

    import torch

    boxes, ncyc, every = 6, 12, 10
    want = []
    for i in range(boxes):
        g = prs.Simulation(dims, N, prec, seed=40 + i)
        g.init(1.0)
        want.append((g.run(ncyc, every), g.copy_out()))
        g.close()
    streams = [torch.cuda.Stream() for _ in range(boxes)]
    sims = [prs.Simulation(dims, N, prec, seed=40 + i, stream=streams[i]) for i in range(boxes)]
    got, errors = [None] * boxes, []

    def drive(i):
        try:
            sims[i].init(1.0)
            got[i] = sims[i].run(ncyc, every)
        except Exception as exc:                                 # pragma: no cover - reported below
            errors.append(exc)

    threads = [threading.Thread(target=drive, args=(i,)) for i in range(boxes)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors
    for i in range(boxes):
        assert got[i] == want[i][0], i
        a = sims[i].copy_out()
        assert a[0].tobytes() == want[i][1][0].tobytes() and a[1].tobytes() == want[i][1][1].tobytes(), i
        sims[i].close()
    assert len({r[-1]["link_count"] for r, _ in want}) > 1      # different seeds, different networks


@pytest.mark.parametrize("prec", [prs.F32, prs.F64])
@pytest.mark.parametrize("N", [64, 128, 256])
@pytest.mark.parametrize("every,ncyc", [(10, 40), (1, 130), (64, 3), (65, 3), (7, 19), (200, 2)])
def test_diagnostics_inside_the_cluster_resident_launches(prec, N, every, ncyc):
    """prs_run with the cluster-resident kernel: the diagnostics passes run inside the step launches (up to 64 steps per
    launch, any cadence: several passes per launch, a pass on a launch's last step, launches without a pass).  Counts
    equal to the oracle's on the GPU path's own snapshots and to prs_diagnostics', the double sum within 1e-10; the fields
    bit-identical to the single-step kernel's; one launch per 64 steps and none for the diagnostics."""
    a = prs.Simulation(2, N, prec, seed=8, era_m=2.0)
    a.set_step_kernel(prs.KERNEL_CLUSTER)
    b = prs.Simulation(2, N, prec, seed=8, era_m=2.0)
    b.set_step_kernel(prs.KERNEL_TILED)
    a.init(1.0)
    b.init(1.0)
    l0 = a.kernel_launches
    got = a.run(ncyc, every)
    assert a.kernel_launches - l0 == (ncyc * every + 63) // 64
    for i in range(ncyc):
        b.step(every)
        want = b.diagnostics()
        assert got[i]["step"] == want["step"] == (i + 1) * every and got[i]["eta"] == want["eta"]
        assert got[i]["link_count"] == want["link_count"] and got[i]["wall_sites"] == want["wall_sites"], i
        assert abs(got[i]["sum_ratio"] - want["sum_ratio"]) <= 1e-10 * max(want["sum_ratio"], 1e-300), i
        if i in (0, ncyc - 1):
            o = ref.diagnostics_of(*b.copy_out())
            assert got[i]["link_count"] == o["link_count"] and got[i]["wall_sites"] == o["wall_sites"]
            assert abs(got[i]["sum_ratio"] - o["sum_ratio"]) <= 1e-10 * max(o["sum_ratio"], 1e-300)
    pa, pb = a.copy_out(), b.copy_out()
    assert pa[0].tobytes() == pb[0].tobytes() and pa[1].tobytes() == pb[1].tobytes()
    if N == 256:                                                # the fall-back for devices without room for 16 CTAs
        c = prs.Simulation(2, N, prec, seed=8, era_m=2.0)
        c.set_step_kernel(prs.KERNEL_CLUSTER)
        c.set_option(binding.OPT_CLUSTER_CTAS, 8)
        c.init(1.0)
        got8 = c.run(ncyc, every)
        assert c.step_launch_info()["grid"] == [8, 1, 1] and a.step_launch_info()["grid"] == [16, 1, 1]
        for x, y in zip(got, got8):
            assert (x["step"], x["link_count"], x["wall_sites"]) == (y["step"], y["link_count"], y["wall_sites"])
            assert abs(x["sum_ratio"] - y["sum_ratio"]) <= 1e-10 * max(y["sum_ratio"], 1e-300)
        pc = c.copy_out()
        assert pa[0].tobytes() == pc[0].tobytes() and pa[1].tobytes() == pc[1].tobytes()
        c.close()
    a.run(2, every)                                             # more cycles after a finished batch continue the count
    again = a.run(1, every)
    b.step(3 * every)
    w = b.diagnostics()
    assert again[0]["step"] == w["step"] and again[0]["link_count"] == w["link_count"]
    a.close()
    b.close()


def test_batched_cycles_error_paths():
    from paper_1710_10420_b200 import sharded

    g = prs.Simulation(2, 64, prs.F32)
    with pytest.raises(prs.PrsError) as e:
        g.run(1, 1)                                             # no state yet
    assert e.value.code == 4
    g.init(1.0)
    with pytest.raises(prs.PrsError) as e:
        g.run(-1, 1)
    assert e.value.code == 1
    s = sharded.SlabSimulation(64, 0, 16, prs.F32)
    s.init(1.0)
    with pytest.raises(prs.PrsError) as e:
        s.run(1, 4)                                             # a slab's halo must be exchanged between passes
    assert e.value.code == 2
