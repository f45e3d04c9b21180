"""Pins of the oracle's initial-condition generator."""
import numpy as np
import pytest

from oracle import binding as ref
from tests.goldenio import read_philox_field_values, read_philox_kat


def test_philox_known_answer_vectors():
    kats = read_philox_kat()
    assert len(kats) == 3
    for ctr, key, want in kats:
        assert ref.philox4x32_10(ctr, key) == want


def test_printed_field_values_pin_the_site_to_counter_and_word_mapping():
    """SURVEY.md Appendix B prints twelve field values (seed 42 sites 0..3 and 20..23 with their words, seed 0
    sites 0..3) and one block on the 64-bit path (seed 2^32+7, q = 2^32+1).  They pin init_value's mapping
    site -> (counter, word, 24-bit shift, scale) against numbers that do not come from this repository's
    code: a swapped word order, an off-by-one shift or a 32-bit truncation of q or of the seed fails here."""
    values, blocks = read_philox_field_values()
    assert len(values) == 12 and len(blocks) == 1
    for seed, site, word, phi in values:
        assert ref.init_value(seed, site, 1.0) == phi, (seed, site)
        assert ref.init_value(seed, site, 1.75) == 1.75 * phi
        if word is not None:                              # the printed word and the printed value agree
            assert (2 * (word >> 8) + 1 - (1 << 24)) / float(1 << 24) == phi
    # a lattice initialised by the oracle holds the same numbers at those sites (FP32 and FP64)
    for prec in (ref.F32, ref.F64):
        for seed in (42, 0):
            sim = ref.RefSim(2, 8, prec, seed=seed)
            sim.init(1.0)
            flat = sim.copy_out()[0].ravel()
            for sd, site, _, phi in values:
                if sd == seed:
                    assert float(flat[site]) == phi
    for seed, q, words in blocks:
        assert q >= 1 << 32 and seed >= 1 << 32
        assert ref.philox4x32_10([q & 0xffffffff, q >> 32, 0, 0], [seed & 0xffffffff, seed >> 32]) == words
        for j, w in enumerate(words):
            assert ref.init_value(seed, 4 * q + j, 1.0) == (2 * (w >> 8) + 1 - (1 << 24)) / float(1 << 24)


def test_philox_is_a_bijection_of_the_counter_on_a_sample():
    # a block cipher in counter mode: distinct counters -> distinct blocks
    seen = set()
    for c0 in range(512):
        seen.add(ref.philox4x32_10([c0, 0, 0, 0], [7, 0]))
    assert len(seen) == 512


def test_site_to_counter_mapping_and_value_formula():
    # site s uses word (s & 3) of the block with counter (s >> 2, 0, 0, 0)... split in 32-bit halves
    for seed in (0, 42, (1 << 32) + 7):
        key = [seed & 0xffffffff, seed >> 32]
        for s in (0, 1, 2, 3, 4, 21, 1023, (1 << 34) + 5, 4 * ((1 << 32) + 1) + 2):
            q = s >> 2
            w = ref.philox4x32_10([q & 0xffffffff, q >> 32, 0, 0], key)[s & 3]
            k = w >> 8
            want = (2 * k + 1 - (1 << 24)) / float(1 << 24)
            assert ref.init_value(seed, s, 1.0) == want
            assert ref.init_value(seed, s, 2.5) == 2.5 * want


def test_values_are_float32_exact_odd_multiples_never_zero_or_one():
    vals = np.array([ref.init_value(5, s) for s in range(4096)])
    assert np.all(vals.astype(np.float32).astype(np.float64) == vals)
    assert np.all(np.abs(vals) < 1.0) and np.all(vals != 0.0)
    ints = vals * (1 << 24)
    assert np.all(ints == np.round(ints)) and np.all(np.abs(ints.astype(np.int64)) % 2 == 1)


def test_uniformity_of_the_initial_field():
    sim = ref.RefSim(2, 256, ref.F64, seed=3)
    sim.init(1.0)
    phi, pd = sim.copy_out()
    assert np.all(pd == 0.0) and not np.any(np.signbit(pd))
    S = phi.size
    # uniform(-1,1): mean 0 +- 1/sqrt(3S), variance 1/3, lag-1 correlation 0
    assert abs(phi.mean()) < 5.0 / np.sqrt(3 * S)
    assert abs(phi.var() - 1.0 / 3.0) < 0.01
    flat = phi.ravel()
    assert abs(np.mean(flat[:-1] * flat[1:])) < 5.0 / (3.0 * np.sqrt(S))
    hist, _ = np.histogram(flat, bins=16, range=(-1, 1))
    assert np.all(np.abs(hist - S / 16) < 6 * np.sqrt(S / 16))


def test_init_matches_value_function_and_precisions_agree():
    a = ref.RefSim(3, 8, ref.F32, seed=11)
    b = ref.RefSim(3, 8, ref.F64, seed=11)
    a.init(1.0)
    b.init(1.0)
    pa, _ = a.copy_out()
    pb, _ = b.copy_out()
    assert np.array_equal(pa.astype(np.float64), pb)
    want = np.array([ref.init_value(11, s) for s in range(512)]).reshape(8, 8, 8)
    assert np.array_equal(pb, want)


def test_different_seeds_differ():
    a = ref.RefSim(2, 16, seed=1)
    b = ref.RefSim(2, 16, seed=2)
    a.init(1.0)
    b.init(1.0)
    assert not np.array_equal(a.copy_out()[0], b.copy_out()[0])


def test_bad_arguments_are_rejected():
    with pytest.raises(RuntimeError):
        ref.RefSim(4, 8)
    with pytest.raises(RuntimeError):
        ref.RefSim(2, 0)
    with pytest.raises(RuntimeError):
        ref.RefSim(2, 8, deta=0.0)
    s = ref.RefSim(2, 8)
    with pytest.raises(RuntimeError):
        s.step(1)            # before init
    with pytest.raises(RuntimeError):
        s.init(0.0)
