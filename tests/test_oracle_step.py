"""Pins of the oracle's step (Eqs. 1, 3-6) against things the paper and mathematics fix.

Each test is chosen so that one plausible mistake (dropped term, wrong sign / index / coefficient,
wrong time level of eta, Gauss-Seidel instead of Jacobi, ...) fails it.  None of them re-types the
oracle's per-site formula: they use exact hand values, closed forms and exact invariants.
"""
import numpy as np
import pytest

from oracle import binding as ref
from tests import fieldgen as fg
from tests.goldenio import as_array, read_sections

PRECS = [(ref.F32, np.float32), (ref.F64, np.float64)]


def run(dims, N, prec, phi, pd, nsteps, eta0=1.0, arith=ref.ARITH_LITERAL, threads=1, **kw):
    sim = ref.RefSim(dims, N, prec, arith=arith, threads=threads, **kw)
    sim.copy_in(phi, pd, eta0=eta0, step=0)
    sim.step(nsteps)
    out = sim.copy_out()
    sim.close()
    return out


# ------------------------------------------------------------------ P1: hand-computed 4x4 step

@pytest.mark.parametrize("prec,dt", PRECS)
@pytest.mark.parametrize("arith", [ref.ARITH_LITERAL, ref.ARITH_COEF, ref.ARITH_FMA])
def test_hand_computed_4x4_step(prec, dt, arith):
    g = read_sections("step_4x4.txt")
    phi0, pd0 = as_array(g["phi0"], dt), as_array(g["phidot0"], dt)
    phi1, pd1 = run(2, 4, prec, phi0, pd0, 1, eta0=3.0, arith=arith,
                    alpha=3.0, era_m=1.0, deta=0.5, W0=np.pi, phi0=1.0)
    want_pd, want_phi = as_array(g["phidot1"]), as_array(g["phi1"])
    # values are O(1): 2 ulp(1) of the type, as the operands of the last few operations are O(1..5)
    tol = 4 * np.finfo(dt).eps
    assert np.max(np.abs(pd1.astype(np.float64) - want_pd)) <= tol * 5
    assert np.max(np.abs(phi1.astype(np.float64) - want_phi)) <= tol * 5
    # the exactly representable entries come out exact (all operands dyadic, no rounding at all)
    assert pd1[0, 0] == -2.0 and phi1[0, 0] == 0.0 and not np.signbit(phi1[0, 0])
    if arith == ref.ARITH_LITERAL:       # A = 3/5 and B = 2/5 are not dyadic, so only the literal form is exact here
        assert phi1[0, 1] == 0.5 and pd1[0, 1] == 0.0


def test_scalars_of_the_hand_example_and_eq6_time_level():
    s = ref.scalars(0, eta0=3.0, alpha=3.0, era_m=1.0, deta=0.5, W0=np.pi, phi0=1.0)
    assert s["delta"] == 0.25 and s["eta"] == 3.0
    assert abs(s["V0"] - 0.5) < 1e-15 and abs(s["K"] - 2.0) < 1e-15 and s["I"] == 1.0
    assert s["A"] == 0.6 and s["B"] == 0.4
    # eta_n = eta0 + n*deta (time level of phi^n), matter era doubles delta
    s5 = ref.scalars(5, eta0=1.0, alpha=3.0, era_m=2.0, deta=0.1)
    assert s5["eta"] == 1.0 + 5 * 0.1
    assert abs(s5["delta"] - 0.5 * 3.0 * 0.1 / 1.5 * 2.0) < 1e-16
    # BASELINE.json: V0 = pi^2 / (2 W0^2) at phi0 = 1, W0 = 10
    s10 = ref.scalars(0)
    assert abs(s10["V0"] - np.pi ** 2 / 200.0) < 1e-17


# ------------------------------------------------------------------ P2: exact fixed points

@pytest.mark.parametrize("prec,dt", PRECS)
@pytest.mark.parametrize("dims,N", [(2, 12), (3, 6)])
@pytest.mark.parametrize("arith", [ref.ARITH_LITERAL, ref.ARITH_COEF, ref.ARITH_FMA])
@pytest.mark.parametrize("era_m", [0.0, 1.0, 2.0])
def test_vacua_are_exact_fixed_points(prec, dt, dims, N, era_m, arith):
    # In the contracted form t = fma(phi^2, 1/phi0^2, -1) is the exact residual of the rounded 1/phi0^2,
    # so the vacuum is an exact fixed point only where 1/phi0^2 is representable (phi0 = 1, 2, ...);
    # the other forms round phi^2 * (1/phi0^2) to exactly 1 for phi0 = 3 as well.
    for sign in (+1.0, -1.0):
        for phi0 in ((1.0, 2.0) if arith == ref.ARITH_FMA else (1.0, 3.0)):
            phi = np.full((N,) * dims, sign * phi0, dt)
            pd = np.zeros_like(phi)
            p, v = run(dims, N, prec, phi, pd, 25, era_m=era_m, phi0=phi0, arith=arith)
            assert np.array_equal(p, phi) and np.all(v == 0)


# ------------------------------------------------------------------ P3-P5: exact symmetries

@pytest.mark.parametrize("prec,dt", PRECS)
@pytest.mark.parametrize("dims,N", [(2, 10), (3, 7)])
@pytest.mark.parametrize("arith", [ref.ARITH_LITERAL, ref.ARITH_COEF, ref.ARITH_FMA])
def test_oddness_is_bit_exact(prec, dt, dims, N, arith):
    phi, pd = fg.random_state(dims, N, 5, dt)
    p1, v1 = run(dims, N, prec, phi, pd, 7, arith=arith)
    p2, v2 = run(dims, N, prec, -phi, -pd, 7, arith=arith)
    assert np.array_equal(p1, -p2) and np.array_equal(v1, -v2)


@pytest.mark.parametrize("prec,dt", PRECS)
@pytest.mark.parametrize("arith", [ref.ARITH_LITERAL, ref.ARITH_COEF, ref.ARITH_FMA])
@pytest.mark.parametrize("dims,N,shift", [(2, 9, (3, -2)), (2, 16, (1, 0)), (3, 6, (1, 2, 5)), (3, 5, (0, 0, 1))])
def test_translation_equivariance_is_bit_exact(prec, dt, dims, N, shift, arith):
    phi, pd = fg.random_state(dims, N, 6, dt)
    p1, v1 = run(dims, N, prec, phi, pd, 5, arith=arith)
    p2, v2 = run(dims, N, prec, fg.roll_state(phi, shift), fg.roll_state(pd, shift), 5, arith=arith)
    assert np.array_equal(fg.roll_state(p1, shift), p2)
    assert np.array_equal(fg.roll_state(v1, shift), v2)


@pytest.mark.parametrize("prec,dt", PRECS)
@pytest.mark.parametrize("arith", [ref.ARITH_LITERAL, ref.ARITH_COEF, ref.ARITH_FMA])
@pytest.mark.parametrize("dims,N", [(2, 8), (3, 6)])
def test_reflection_equivariance_is_bit_exact(prec, dt, dims, N, arith):
    phi, pd = fg.random_state(dims, N, 7, dt)
    p1, v1 = run(dims, N, prec, phi, pd, 5, arith=arith)
    for ax in range(dims):
        p2, v2 = run(dims, N, prec, fg.flip_axis(phi, ax), fg.flip_axis(pd, ax), 5, arith=arith)
        assert np.array_equal(fg.flip_axis(p1, ax), p2) and np.array_equal(fg.flip_axis(v1, ax), v2)


@pytest.mark.parametrize("arith", [ref.ARITH_LITERAL, ref.ARITH_COEF, ref.ARITH_FMA])
@pytest.mark.parametrize("prec,dt", PRECS)
def test_2d_transpose_equivariance_is_bit_exact(prec, dt, arith):
    phi, pd = fg.random_state(2, 11, 8, dt)
    p1, v1 = run(2, 11, prec, phi, pd, 5, arith=arith)
    p2, v2 = run(2, 11, prec, np.ascontiguousarray(phi.T), np.ascontiguousarray(pd.T), 5, arith=arith)
    assert np.array_equal(p1.T, p2) and np.array_equal(v1.T, v2)


@pytest.mark.parametrize("prec,dt", PRECS)
def test_3d_field_uniform_in_z_reproduces_the_2d_run_up_to_rounding(prec, dt):
    # (sx+sy)+(c+c)-6c versus (sx+sy)-4c: equal in exact arithmetic, so the 3D run of a z-uniform field
    # must track the 2D run; pins the z-terms of the 7-point stencil (a missing/extra z term shows)
    N = 8
    phi2, pd2 = fg.random_state(2, N, 9, dt)
    phi3 = np.ascontiguousarray(np.broadcast_to(phi2, (N, N, N)))
    pd3 = np.ascontiguousarray(np.broadcast_to(pd2, (N, N, N)))
    p2, v2 = run(2, N, prec, phi2, pd2, 10)
    p3, v3 = run(3, N, prec, phi3, pd3, 10)
    for z in range(N):
        assert np.array_equal(p3[z], p3[0])
    tol = 200 * np.finfo(dt).eps
    assert np.max(np.abs(p3[0].astype(np.float64) - p2)) < tol
    assert np.max(np.abs(v3[0].astype(np.float64) - v2)) < tol


# ------------------------------------------------------------------ Jacobi, threads, arithmetic modes

@pytest.mark.parametrize("prec,dt", PRECS)
def test_single_spike_spreads_exactly_one_site_per_step(prec, dt):
    # Jacobi update ("embarrassingly parallel steps"): after one step only the spike and its
    # 2d neighbours differ from the vacuum; a Gauss-Seidel sweep would smear further along the sweep.
    N = 9
    phi = np.ones((N, N, N), dt)
    phi[4, 4, 4] = 0.25
    pd = np.zeros_like(phi)
    p, v = run(3, N, prec, phi, pd, 1)
    changed = np.argwhere(p != 1.0)
    dist = np.abs(changed - 4).sum(axis=1)
    assert len(changed) == 7 and dist.max() == 1
    # the six neighbours got exactly deta * deta/(1+delta) * (0.25 - 1) from the Laplacian, same value
    nb = [p[3, 4, 4], p[5, 4, 4], p[4, 3, 4], p[4, 5, 4], p[4, 4, 3], p[4, 4, 5]]
    assert len(set(float(x) for x in nb)) == 1
    delta = 0.5 * 3.0 * 0.1
    want = 1.0 + 0.1 * (0.1 * (0.25 - 1.0)) / (1.0 + delta)
    assert abs(float(nb[0]) - want) < 4 * np.finfo(dt).eps


@pytest.mark.parametrize("prec,dt", PRECS)
@pytest.mark.parametrize("dims,N", [(2, 33), (3, 12)])
def test_threads_do_not_change_a_bit(prec, dt, dims, N):
    phi, pd = fg.random_state(dims, N, 10, dt)
    a = run(dims, N, prec, phi, pd, 6, threads=1)
    b = run(dims, N, prec, phi, pd, 6, threads=4)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


@pytest.mark.parametrize("prec,dt,tol", [(ref.F32, np.float32, 2e-6), (ref.F64, np.float64, 4e-15)])
@pytest.mark.parametrize("dims,N", [(2, 32), (3, 10)])
def test_coef_fma_and_literal_arithmetic_agree_to_rounding(prec, dt, tol, dims, N):
    phi, _ = fg.random_state(dims, N, 11, dt)
    pd = np.zeros_like(phi)
    a = run(dims, N, prec, phi, pd, 20, arith=ref.ARITH_LITERAL)
    for other in (ref.ARITH_COEF, ref.ARITH_FMA):
        b = run(dims, N, prec, phi, pd, 20, arith=other)
        assert np.max(np.abs(a[0].astype(np.float64) - b[0])) < tol
        assert np.max(np.abs(a[1].astype(np.float64) - b[1])) < tol
        assert not (np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]))   # the forms do round differently


def test_step_counter_and_eta_advance_without_accumulation():
    sim = ref.RefSim(2, 4, ref.F64, deta=0.1)
    sim.init(1.0)
    sim.step(3)
    sim.step(4)
    d = sim.diagnostics()
    assert d["step"] == 7 and d["eta"] == 1.0 + 7 * 0.1
    # stepping 3+4 equals stepping 7
    sim2 = ref.RefSim(2, 4, ref.F64, deta=0.1)
    sim2.init(1.0)
    sim2.step(7)
    assert np.array_equal(sim.copy_out()[0], sim2.copy_out()[0])


def test_step_sites_helper_matches_full_step():
    for dims, N in ((2, 9), (3, 6)):
        for prec, dt in PRECS:
            phi, pd = fg.random_state(dims, N, 12, dt)
            sim = ref.RefSim(dims, N, prec, era_m=2.0)
            sim.copy_in(phi, pd, eta0=1.0, step=4)
            sim.step(1)
            p1, v1 = sim.copy_out()
            sites = np.arange(phi.size)
            po, vo = ref.step_sites(phi, pd, sites, n=4, eta0=1.0, era_m=2.0)
            assert np.array_equal(po, p1.ravel()) and np.array_equal(vo, v1.ravel())


# ------------------------------------------------------------------ P6: uniform field = scalar ODE

@pytest.mark.parametrize("dims,N", [(2, 6), (3, 5)])
def test_uniform_field_follows_the_scalar_recurrence(dims, N):
    # lap == 0 exactly for a uniform field; the remaining scalar recurrence is evaluated here with
    # python floats written in the paper's own form (Eq. 4 literally, one division)
    c0, v0, deta, eta0, alpha, m, W0 = 0.3, 0.05, 0.1, 1.0, 3.0, 1.0, 10.0
    V0 = np.pi ** 2 / (2 * W0 ** 2)
    phi = np.full((N,) * dims, c0)
    pd = np.full((N,) * dims, v0)
    p, v = run(dims, N, ref.F64, phi, pd, 40, eta0=eta0)
    c, w = c0, v0
    for n in range(40):
        delta = 0.5 * alpha * deta / (eta0 + n * deta) * m
        dV = 4 * V0 * c * (c * c - 1.0)
        w = ((1 - delta) * w - deta * dV) / (1 + delta)
        c = c + deta * w
    assert np.all(p == p.flat[0]) and np.all(v == v.flat[0])
    assert abs(p.flat[0] - c) < 1e-14 and abs(v.flat[0] - w) < 1e-14


# ------------------------------------------------------------------ the scale-factor exponent beta of Eq. 2

def test_beta_scalars_closed_form():
    # a = (eta/eta0)^m with a(eta0) = 1; K_n = (4 V0 / phi0^2) * a^beta.  eta0 = 1, deta = 1/2, n = 6 ->
    # eta = 4; m = 2, beta = 2 -> a^beta = 4^4 = 256 exactly; W0 = pi -> 4 V0 = 2.
    s = ref.scalars(6, eta0=1.0, alpha=2.0, era_m=2.0, deta=0.5, W0=np.pi, phi0=1.0, beta=2.0)
    assert s["eta"] == 4.0 and s["K"] == 512.0 and s["delta"] == 0.5 * 2.0 * (0.5 / 4.0) * 2.0
    assert ref.scalars(6, era_m=2.0, deta=0.5, W0=np.pi, beta=0.0)["K"] == 2.0          # PRS: no factor
    assert ref.scalars(6, era_m=0.0, deta=0.5, W0=np.pi, beta=2.0)["K"] == 2.0          # no expansion: a = 1
    assert ref.scalars(0, eta0=3.0, era_m=1.0, deta=0.5, W0=np.pi, beta=2.0)["K"] == 2.0  # a(eta0) = 1


@pytest.mark.parametrize("arith", [ref.ARITH_LITERAL, ref.ARITH_COEF, ref.ARITH_FMA])
def test_beta_zero_changes_nothing_and_beta_two_does(arith):
    phi, pd = fg.random_state(3, 6, 31, np.float64)
    a = run(3, 6, ref.F64, phi, pd, 10, arith=arith)
    b = run(3, 6, ref.F64, phi, pd, 10, arith=arith, beta=0.0)
    c = run(3, 6, ref.F64, phi, pd, 10, arith=arith, alpha=2.0, beta=2.0)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    assert not np.array_equal(a[0], c[0])


@pytest.mark.parametrize("dims,N", [(2, 6), (3, 5)])
@pytest.mark.parametrize("alpha,beta,m", [(2.0, 2.0, 1.0), (2.0, 2.0, 2.0), (3.0, 1.0, 2.0)])
def test_uniform_field_follows_the_scalar_recurrence_with_the_scale_factor(dims, N, alpha, beta, m):
    # as P6, with dV/dphi multiplied by a^beta = (eta_n/eta0)^(m beta) (Eq. 2, :34-36)
    c0, v0, deta, eta0, W0 = 0.3, 0.05, 0.1, 2.0, 10.0
    V0 = np.pi ** 2 / (2 * W0 ** 2)
    phi = np.full((N,) * dims, c0)
    pd = np.full((N,) * dims, v0)
    p, v = run(dims, N, ref.F64, phi, pd, 40, eta0=eta0, alpha=alpha, era_m=m, beta=beta)
    c, w = c0, v0
    for n in range(40):
        eta = eta0 + n * deta
        delta = 0.5 * alpha * deta / eta * m
        dV = (eta / eta0) ** (m * beta) * 4 * V0 * c * (c * c - 1.0)
        w = ((1 - delta) * w - deta * dV) / (1 + delta)
        c = c + deta * w
    assert np.all(p == p.flat[0]) and np.all(v == v.flat[0])
    assert abs(p.flat[0] - c) < 1e-13 and abs(v.flat[0] - w) < 1e-13


# ------------------------------------------------------------------ P7: free discrete wave (exact eigenmode)

def _lattice_k2(N, modes):
    return sum((2.0 * np.sin(np.pi * m / N)) ** 2 for m in modes)


@pytest.mark.parametrize("dims,N,modes", [(2, 32, (3, 0)), (2, 32, (0, 5)), (2, 24, (2, 7)),
                                          (3, 16, (1, 0, 0)), (3, 16, (0, 0, 3)), (3, 12, (2, 1, 5))])
def test_free_plane_wave_obeys_the_exact_lattice_dispersion(dims, N, modes):
    deta, nsteps = 0.1, 200
    lam = _lattice_k2(N, modes)
    omega = 2.0 / deta * np.arcsin(0.5 * deta * np.sqrt(lam))     # sin^2(w deta/2) = deta^2 lam / 4
    phi0 = fg.plane_wave(dims, N, modes)
    phim1 = fg.plane_wave(dims, N, modes, phase=+omega * deta)    # phi^{-1}
    pd = (phi0 - phim1) / deta                                     # phidot^{-1/2}
    p, v = run(dims, N, ref.F64, phi0, pd, nsteps, era_m=0.0, deta=deta, W0=1e9)
    want = fg.plane_wave(dims, N, modes, phase=-omega * deta * nsteps)
    want_prev = fg.plane_wave(dims, N, modes, phase=-omega * deta * (nsteps - 1))
    assert np.max(np.abs(p - want)) < 2e-12
    assert np.max(np.abs(v - (want - want_prev) / deta)) < 2e-11


# ------------------------------------------------------------------ P8: small oscillations about the vacuum

@pytest.mark.parametrize("dims,N,modes,W0,phi0", [(2, 32, (0, 0), 10.0, 1.0), (2, 32, (2, 1), 10.0, 1.0),
                                                  (3, 12, (1, 2, 0), 10.0, 1.0), (2, 16, (1, 3), 5.0, 2.0),
                                                  (3, 8, (0, 0, 0), 4.0, 0.5)])
def test_massive_dispersion_about_the_vacuum(dims, N, modes, W0, phi0):
    # Klein-Gordon about phi0: Omega^2 = M^2 + sum (2 sin(k/2))^2 with M^2 = V''(phi0) = 8 V0/phi0^2
    # = (2 pi / W0)^2 for V0 = pi^2 phi0^2 / (2 W0^2).  Pins the potential's coefficient and the
    # relative sign of Laplacian and dV/dphi in Eq. 4.
    deta, nsteps, eps = 0.1, 150, 1e-7
    M2 = (2.0 * np.pi / W0) ** 2
    Om = 2.0 / deta * np.arcsin(0.5 * deta * np.sqrt(M2 + _lattice_k2(N, modes)))
    f0 = fg.plane_wave(dims, N, modes, amp=eps)
    fm1 = fg.plane_wave(dims, N, modes, phase=+Om * deta, amp=eps)
    p, v = run(dims, N, ref.F64, phi0 + f0, (f0 - fm1) / deta, nsteps, era_m=0.0, deta=deta, W0=W0, phi0=phi0)
    want = fg.plane_wave(dims, N, modes, phase=-Om * deta * nsteps, amp=eps)
    # linearisation error is O(eps^2 t) ~ 1e-13 and rounding of phi0+x is ~1e-16: both << 1e-4*eps
    assert np.max(np.abs((p - phi0) - want)) < 1e-4 * eps


# ------------------------------------------------------------------ damping: exact discrete Abel identity

@pytest.mark.parametrize("dims,N", [(2, 16), (3, 8)])
@pytest.mark.parametrize("alpha,era_m,eta0", [(3.0, 1.0, 1.0), (3.0, 2.0, 1.0), (2.0, 1.0, 2.5)])
def test_wronskian_decays_by_the_product_of_eq6_factors(dims, N, alpha, era_m, eta0):
    # For the linear part of Eqs. 3-5 (potential switched off by W0 -> inf) two solutions x, y satisfy
    #   W_n = sum_s (x_s vy_s - y_s vx_s),  W_{n+1} = W_n (1-delta_n)/(1+delta_n)   exactly,
    # because the Laplacian is symmetric.  Pins Eq. 4's damping structure and Eq. 6 (alpha, era, eta_n).
    deta, nsteps = 0.1, 60
    x0, vx0 = fg.random_state(dims, N, 21, np.float64)
    y0, vy0 = fg.random_state(dims, N, 22, np.float64)
    kw = dict(eta0=eta0, alpha=alpha, era_m=era_m, deta=deta, W0=1e9)
    x1, vx1 = run(dims, N, ref.F64, x0, vx0, nsteps, **kw)
    y1, vy1 = run(dims, N, ref.F64, y0, vy0, nsteps, **kw)
    W_0 = np.sum(x0 * vy0 - y0 * vx0)
    W_1 = np.sum(x1 * vy1 - y1 * vx1)
    prod = 1.0
    for n in range(nsteps):
        d = 0.5 * alpha * deta / (eta0 + n * deta) * era_m
        prod *= (1 - d) / (1 + d)
    assert abs(W_1 / W_0 - prod) < 1e-10 * abs(prod) + 1e-13


def test_undamped_run_conserves_the_wronskian_and_is_time_reversible():
    x0, vx0 = fg.random_state(2, 12, 31, np.float64)
    p, v = run(2, 12, ref.F64, x0, vx0, 50, era_m=0.0)
    # leapfrog with delta = 0 is exactly reversible up to rounding: run back with phidot -> -phidot.
    # state (phi^n, phidot^{n-1/2}); reversed state is (phi^n, -phidot^{n+1/2}); one extra half step
    # bookkeeping: phi^{n-1} = phi^n - deta*phidot^{n-1/2}
    back_phi = p - 0.1 * v            # phi^{n-1}
    bp, bv = run(2, 12, ref.F64, back_phi, -v, 49, era_m=0.0)   # reaches phi^0
    assert np.max(np.abs(bp - x0)) < 1e-12


@pytest.mark.parametrize("era_m,power", [(1.0, -1.5), (2.0, -3.0)])
def test_damping_envelope_follows_the_friction_power_law(era_m, power):
    # energy-like envelope of a k=0 vacuum oscillation decays as (eta/eta0)^(-alpha m / 2) in amplitude
    N, deta, eta0, eps = 4, 0.1, 1.0, 1e-3
    phi = np.full((N, N), 1.0 + eps)
    pd = np.zeros_like(phi)
    sim = ref.RefSim(2, N, ref.F64, era_m=era_m, deta=deta)
    sim.copy_in(phi, pd, eta0=eta0, step=0)
    M = 2 * np.pi / 10.0
    amps, etas = [], []
    for n in range(1, 1500):
        sim.step(1)
        p, v = sim.copy_out()
        x, w = p.flat[0] - 1.0, v.flat[0]
        amps.append(np.sqrt(x * x + (w / M) ** 2))
        etas.append(eta0 + n * deta)
    amps, etas = np.array(amps), np.array(etas)
    sel = etas > 20
    slope = np.polyfit(np.log(etas[sel]), np.log(amps[sel]), 1)[0]
    assert abs(slope - power) < 0.05


# ------------------------------------------------------------------ P9: planar kink pair

@pytest.mark.parametrize("dims,N", [(2, 64), (3, 32)])
@pytest.mark.parametrize("era_m", [0.0, 1.0])
def test_static_kink_pair_stays_put(dims, N, era_m):
    W0 = 10.0 if N >= 64 else 5.0
    kappa = np.pi / W0                                   # sqrt(2 V0)/phi0
    phi = fg.kink_pair(dims, N, kappa)
    phi = 0.5 * (phi + phi[..., ::-1])                   # exact mirror symmetry about x = (N-1)/2
    pd = np.zeros_like(phi)
    sim = ref.RefSim(dims, N, ref.F64, era_m=era_m, W0=W0)
    sim.copy_in(phi, pd, eta0=1.0, step=0)
    sign0 = np.signbit(phi)
    for _ in range(10):
        sim.step(40)
        p, v = sim.copy_out()
        d = sim.diagnostics()
        assert d["link_count"] == 2 * N ** (dims - 1)
        assert d["wall_sites"] == 4 * N ** (dims - 1)
        assert np.array_equal(np.signbit(p), sign0)      # walls stay centred between the same sites
        assert np.array_equal(p, p[..., ::-1])           # mirror symmetry preserved bit-exactly
        assert np.max(np.abs(v)) < 0.05 * kappa          # |phidot| ~ kappa*v: lattice relaxation only, v < 5% of c
        # uniform along the wall
        assert np.array_equal(p, np.broadcast_to(p[(0,) * (dims - 1)], p.shape))


# ------------------------------------------------------------------ P10 (dynamics part): boosted kink

def test_boosted_kink_pair_moves_at_its_velocity():
    N, W0, vel, deta = 256, 10.0, 0.4, 0.1
    kappa, gamma = np.pi / W0, 1.0 / np.sqrt(1 - 0.4 ** 2)
    # walls approach each other: left wall moves right (+v), right wall moves left
    phi_now = fg.kink_pair(2, N, kappa, gamma=gamma, shift=0.0)
    phi_prev = fg.kink_pair(2, N, kappa, gamma=gamma, shift=-vel * deta)
    pd = (phi_now - phi_prev) / deta
    sim = ref.RefSim(2, N, ref.F64, era_m=0.0, deta=deta, W0=W0)
    sim.copy_in(phi_now, pd, eta0=1.0, step=0)
    nsteps = 500                                         # t = 50 -> each wall moves 20 sites
    sim.step(nsteps)
    p, v = sim.copy_out()
    row = p[0]
    cross = np.where(np.signbit(row[:-1]) != np.signbit(row[1:]))[0]
    assert len(cross) == 2
    # sub-site zero crossing by linear interpolation
    pos = [i + row[i] / (row[i] - row[i + 1]) for i in cross]
    x1, x2 = N / 4 - 0.5 + vel * deta * nsteps, 3 * N / 4 - 0.5 - vel * deta * nsteps
    assert abs(pos[0] - x1) < 0.5 and abs(pos[1] - x2) < 0.5
    d = sim.diagnostics()
    assert abs(d["gv2"] - (gamma * vel) ** 2) < 0.05 * (gamma * vel) ** 2


# ------------------------------------------------------------------ P14: scaling (soft, physics)

def test_network_approaches_scaling_in_a_256_box():
    sim = ref.RefSim(2, 256, ref.F32, seed=1, threads=4)
    sim.init(1.0)
    etas, rhos = [], []
    for _ in range(127):
        sim.step(10)
        d = sim.diagnostics()
        etas.append(d["eta"])
        rhos.append(d["rho"])
    etas, rhos = np.array(etas), np.array(rhos)
    sel = etas >= 13.2                                   # ln(eta) > 2.58
    mu = np.polyfit(np.log(etas[sel]), np.log(rhos[sel]), 1)[0]
    assert -1.25 < mu < -0.7                             # Eq. 9: mu -> -1 (Table I: -0.94 at 2048^2)
    assert rhos[0] > 10 * rhos[-1]
