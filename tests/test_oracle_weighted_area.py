"""Pins of the oracle's orientation-weighted wall area (Eq. 7 as printed, :59-62; reading R15 of
DESIGN.md for where on a link the gradient is taken).  None of these re-types the oracle's loops: an
independent vectorised numpy recount, exact special cases, bounds and closed forms."""
import numpy as np
import pytest

from oracle import binding as ref
from tests import fieldgen as fg


def numpy_weighted_area(phi):
    """Independent recount with whole-array rolls: axis a of the array <-> lattice axis d-1-a."""
    p = phi.astype(np.float64)
    d = p.ndim
    neg = np.signbit(phi)
    total = 0.0
    for k in range(d):                                   # forward links along array axis k
        other = np.roll(p, -1, axis=k)
        cross = neg != np.roll(neg, -1, axis=k)
        g2 = (other - p) ** 2
        gabs = np.abs(other - p)
        for t in range(d):
            if t == k:
                continue
            cen = (np.roll(p, -1, axis=t) - np.roll(p, 1, axis=t)) / 2.0
            gt = (cen + np.roll(cen, -1, axis=k)) / 2.0
            g2 = g2 + gt ** 2
            gabs = gabs + np.abs(gt)
        with np.errstate(invalid="ignore", divide="ignore"):
            w = np.where(gabs == 0.0, 1.0, np.sqrt(g2) / gabs)
        total += float(np.sum(w[cross]))
    return total


@pytest.mark.parametrize("dt", [np.float32, np.float64])
@pytest.mark.parametrize("dims,N,seed", [(2, 8, 1), (2, 13, 2), (3, 6, 3), (3, 9, 4), (2, 2, 5), (3, 2, 6), (2, 1, 7)])
def test_random_fields_against_an_independent_numpy_recount(dims, N, seed, dt):
    phi, _ = fg.random_state(dims, N, seed, dt)
    got, want = ref.weighted_area_of(phi), numpy_weighted_area(phi)
    assert abs(got - want) <= 1e-12 * max(want, 1.0)


@pytest.mark.parametrize("dims,N", [(2, 16), (3, 10)])
def test_bounds_between_count_over_sqrt_d_and_count(dims, N):
    phi, pd = fg.random_state(dims, N, 11, np.float64)
    C = ref.diagnostics_of(phi, pd)["link_count"]
    A = ref.weighted_area_of(phi)
    assert C / np.sqrt(dims) - 1e-9 <= A <= C + 1e-9 and C > 0


@pytest.mark.parametrize("dims", [2, 3])
def test_walls_normal_to_an_axis_have_weight_exactly_one(dims):
    N = 32
    phi = fg.kink_pair(dims, N, np.pi / 10.0, dtype=np.float64)      # uniform across the wall
    assert ref.weighted_area_of(phi) == 2.0 * N ** (dims - 1)
    # ... whichever axis the wall is normal to
    assert ref.weighted_area_of(np.ascontiguousarray(np.moveaxis(phi, -1, 0))) == 2.0 * N ** (dims - 1)


def test_diagonal_wall_in_2d_has_weight_one_over_sqrt_two():
    # phi = cos(2 pi (x + y) / N): near its zeros the profile is linear with equal x and y slopes, so
    # every crossing link weighs 1/sqrt(2) up to O((2 pi / N)^2).
    N = 256
    phi = fg.plane_wave(2, N, (1, 1))
    C = ref.diagnostics_of(phi, np.zeros_like(phi))["link_count"]
    A = ref.weighted_area_of(phi)
    assert C == 4 * N                                               # two zero lines, each cut by N x-links and N y-links
    assert abs(A / C - 1.0 / np.sqrt(2.0)) < 1e-3


def test_body_diagonal_wall_in_3d_has_weight_one_over_sqrt_three():
    N = 96
    phi = fg.plane_wave(3, N, (1, 1, 1))
    C = ref.diagnostics_of(phi, np.zeros_like(phi))["link_count"]
    A = ref.weighted_area_of(phi)
    assert abs(A / C - 1.0 / np.sqrt(3.0)) < 2e-3


@pytest.mark.parametrize("dims,N", [(2, 12), (3, 7)])
def test_invariant_under_negation_translation_reflection(dims, N):
    phi, _ = fg.random_state(dims, N, 21, np.float64)
    A = ref.weighted_area_of(phi)
    for other in (-phi, fg.roll_state(phi, (3, 1, 2)[:dims]), fg.flip_axis(phi, 0), fg.flip_axis(phi, dims - 1)):
        assert abs(ref.weighted_area_of(other) - A) <= 1e-12 * A
    if dims == 2:
        assert abs(ref.weighted_area_of(np.ascontiguousarray(phi.T)) - A) <= 1e-12 * A


def test_single_flipped_site_by_hand():
    # 2D, phi = +1 with one site -1/2: 4 crossing links.  For the x-link from the site to its right
    # neighbour: along g = 1 - (-1/2) = 3/2; across, the central differences vanish at both ends
    # (the neighbours above and below each end are equal), so the weight is 1; same for all four.
    phi = np.ones((6, 6))
    phi[2, 3] = -0.5
    assert ref.weighted_area_of(phi) == 4.0
    # two diagonal neighbours flipped: the x-link right of (2,3) now has a transverse component
    phi[3, 4] = -0.5
    # link (y=2,x=3)->(2,4): along 3/2; across: centre end (phi[3,3]-phi[1,3])/2 = 0, far end
    # (phi[3,4]-phi[1,4])/2 = -3/4, mean -3/8: weight = sqrt(9/4 + 9/64) / (3/2 + 3/8)
    w = np.sqrt(9 / 4 + 9 / 64) / (3 / 2 + 3 / 8)
    assert abs(ref.weighted_area_of(phi) - (4.0 + 4.0 * w)) < 1e-14   # by symmetry four links see a diagonal neighbour
