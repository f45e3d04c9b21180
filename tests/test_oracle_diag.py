"""Pins of the oracle's diagnostics (Eq. 7 link count, Eq. 8 wall velocity)."""
from fractions import Fraction

import numpy as np
import pytest

from oracle import binding as ref
from tests import fieldgen as fg
from tests.goldenio import as_array, read_sections


def brute_links(phi):
    """Recount written differently from the oracle: enumerate the set of undirected nearest-neighbour
    links (as index pairs, multiplicity kept for N=2 where both links join the same pair) and test the
    sign of each; a site is a wall site if it appears in any crossing link."""
    dims, N = phi.ndim, phi.shape[0]
    neg = np.signbit(phi)
    links = []
    for idx in np.ndindex(*phi.shape):
        for ax in range(dims):
            j = list(idx)
            j[ax] = (j[ax] + 1) % N
            links.append((idx, tuple(j)))
    crossing = [(a, b) for a, b in links if neg[a] != neg[b]]
    wall = set()
    for a, b in crossing:
        wall.add(a)
        wall.add(b)
    return len(crossing), wall


def test_hand_example_diagnostics_before_and_after():
    g = read_sections("step_4x4.txt")
    phi0, pd0 = as_array(g["phi0"]), as_array(g["phidot0"])
    C, Nw, S = g["diag0"][0]
    d = ref.diagnostics_of(phi0, pd0, W0=np.pi, phi0=1.0)
    assert d["link_count"] == C and d["wall_sites"] == Nw
    assert abs(d["sum_ratio"] - float(S)) < 1e-13
    assert abs(d["gv2"] - float(S / (2 * Nw))) < 1e-14
    assert d["rho"] == float(Fraction(int(C), 16))
    # after the step phi(0,0) = +0 exactly: positive under the sign-bit rule -> 16 links, not 15
    sim = ref.RefSim(2, 4, ref.F64, alpha=3.0, era_m=1.0, deta=0.5, W0=np.pi)
    sim.copy_in(phi0, pd0, eta0=3.0, step=0)
    sim.step(1)
    d1 = sim.diagnostics()
    C1, Nw1 = g["diag1_counts"][0]
    assert d1["link_count"] == C1 and d1["wall_sites"] == Nw1
    assert d1["step"] == 1 and d1["eta"] == 3.5
    # independent evaluation of sum_ratio from the exact rationals of the fixture
    S1 = sum(v * v / (Fraction(1, 2) * (p * p - 1) ** 2)
             for prow, vrow in zip(g["phi1"], g["phidot1"]) for p, v in zip(prow, vrow) if p * p != 1)
    assert abs(d1["sum_ratio"] - float(S1)) < 1e-12


@pytest.mark.parametrize("dims,N", [(2, 4), (3, 4), (2, 7), (3, 5)])
def test_single_flipped_site(dims, N):
    phi = np.ones((N,) * dims)
    phi[(1,) * dims] = -0.5
    pd = np.full_like(phi, 0.2)
    d = ref.diagnostics_of(phi, pd, W0=10.0)
    assert d["link_count"] == 2 * dims and d["wall_sites"] == 2 * dims + 1
    # the 2d neighbours sit at the vacuum: V = 0 -> contribute 0; only the flipped site counts
    V0 = np.pi ** 2 / 200.0
    want = 0.2 ** 2 / (V0 * (0.25 - 1.0) ** 2)
    assert abs(d["sum_ratio"] - want) < 1e-13 * want
    assert abs(d["gv2"] - want / (2 * (2 * dims + 1))) < 1e-14


@pytest.mark.parametrize("dims,N,seed", [(2, 8, 1), (2, 5, 2), (3, 6, 3), (3, 3, 4), (2, 2, 5), (3, 2, 6), (2, 1, 7)])
@pytest.mark.parametrize("dt", [np.float32, np.float64])
def test_random_fields_against_brute_force(dims, N, seed, dt):
    phi, pd = fg.random_state(dims, N, seed, dt)
    d = ref.diagnostics_of(phi, pd, W0=10.0, phi0=1.0)
    C, wall = brute_links(phi)
    assert d["link_count"] == C and d["wall_sites"] == len(wall)
    V0 = np.pi ** 2 / 200.0
    terms = []
    for idx in wall:
        p, v = float(phi[idx]), float(pd[idx])
        V = V0 * (p * p - 1.0) ** 2
        terms.append(v * v / V if V != 0 else 0.0)
    want = float(np.sum(np.sort(np.array(terms)))) if terms else 0.0
    assert abs(d["sum_ratio"] - want) <= 1e-12 * max(1.0, want)
    assert d["rho"] == C / float(N ** dims)


def test_sign_bit_convention_for_zeros():
    # +0 is positive, -0 is negative (reading G6)
    phi = np.array([[1.0, 0.0], [1.0, 1.0]])
    assert ref.diagnostics_of(phi, np.zeros_like(phi))["link_count"] == 0
    phi[0, 1] = -0.0
    d = ref.diagnostics_of(phi, np.zeros_like(phi))
    assert d["link_count"] == 4 and d["wall_sites"] == 3          # N=2: both links of a pair counted; (1,0) untouched
    # float32 product underflow: a*b < 0 would miss this link, the sign bit does not
    tiny = np.array([[1e-30, -1e-30, 1.0, 1.0]] * 4, np.float32)
    assert ref.diagnostics_of(tiny, np.zeros_like(tiny))["link_count"] == 8


@pytest.mark.parametrize("dims,N", [(2, 9), (3, 5)])
def test_counts_invariant_under_negation_translation_reflection(dims, N):
    phi, pd = fg.random_state(dims, N, 17, np.float64)
    d0 = ref.diagnostics_of(phi, pd)
    variants = [(-phi, -pd), (fg.roll_state(phi, (2,) * dims), fg.roll_state(pd, (2,) * dims)),
                (fg.flip_axis(phi, 0), fg.flip_axis(pd, 0)), (fg.flip_axis(phi, dims - 1), fg.flip_axis(pd, dims - 1))]
    for p, v in variants:
        d = ref.diagnostics_of(p, v)
        assert d["link_count"] == d0["link_count"] and d["wall_sites"] == d0["wall_sites"]
        assert abs(d["sum_ratio"] - d0["sum_ratio"]) < 1e-10 * d0["sum_ratio"]


def test_vacuum_has_no_walls():
    phi = np.full((6, 6, 6), -1.0)
    d = ref.diagnostics_of(phi, np.zeros_like(phi))
    assert d["link_count"] == 0 and d["wall_sites"] == 0 and d["gv2"] == 0.0 and d["sum_ratio"] == 0.0


@pytest.mark.parametrize("dims", [2, 3])
def test_planar_walls_have_area_density_two_over_n(dims):
    # two flat walls normal to x: A = 2 N^(d-1), rho = A/V = 2/N -- links counted == true area
    N = 16
    for axis in range(dims):
        phi = np.moveaxis(fg.kink_pair(dims, N, 0.5), dims - 1, dims - 1 - axis)
        phi = np.ascontiguousarray(phi)
        d = ref.diagnostics_of(phi, np.zeros_like(phi))
        assert d["link_count"] == 2 * N ** (dims - 1)
        assert d["rho"] == 2.0 / N


@pytest.mark.parametrize("vel", [0.1, 0.5, 0.9])
@pytest.mark.parametrize("dims", [2, 3])
def test_eq8_on_an_exact_boosted_kink_snapshot(vel, dims):
    # P10: phi = phi0 tanh(g k (x - v t)), phidot = -g k v phi0 sech^2(...) at the same instant gives
    # phidot^2 / V = 2 g^2 v^2 at every site, so (gamma v)^2 of Eq. 8 = g^2 v^2 exactly: pins E_k =
    # phidot^2, the 1/(2N) factor and V(phi) with V0 = pi^2 phi0^2 / (2 W0^2).
    N, W0, phi0 = 32, 6.0, 1.5
    kappa, gamma = np.pi / W0, 1.0 / np.sqrt(1.0 - vel * vel)
    x = np.arange(N, dtype=np.float64)
    x1, x2 = N / 4 - 0.5, 3 * N / 4 - 0.5
    u1, u2 = gamma * kappa * (x - x1), gamma * kappa * (x - x2)
    prof = phi0 * np.where(x < N / 2, np.tanh(u1), -np.tanh(u2))
    vprof = np.where(x < N / 2, -gamma * kappa * vel * phi0 / np.cosh(u1) ** 2,
                     +gamma * kappa * vel * phi0 / np.cosh(u2) ** 2)
    phi = np.ascontiguousarray(np.broadcast_to(prof, (N,) * dims))
    pd = np.ascontiguousarray(np.broadcast_to(vprof, (N,) * dims))
    d = ref.diagnostics_of(phi, pd, W0=W0, phi0=phi0)
    assert d["wall_sites"] == 4 * N ** (dims - 1)
    assert abs(d["gv2"] - (gamma * vel) ** 2) < 1e-9 * (gamma * vel) ** 2


def test_float32_snapshot_uses_double_for_the_ratio():
    phi, pd = fg.random_state(3, 6, 23, np.float32)
    a = ref.diagnostics_of(phi, pd)
    b = ref.diagnostics_of(phi.astype(np.float64), pd.astype(np.float64))
    assert a["link_count"] == b["link_count"] and a["wall_sites"] == b["wall_sites"]
    assert a["sum_ratio"] == b["sum_ratio"]
