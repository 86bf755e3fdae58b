"""Pins of oracle/rng_oracle.py (the field sampler of the propagation step; Eq. 4's "p(x) is the normal distribution",
PAPER.md:74-79).  The generator is Philox4x32-10 restated from the published algorithm; what fixes it here, other than
itself: the known-answer vectors published with the algorithm (Random123's kat_vectors for philox4x32 with 10 rounds),
the range and grid of the uniforms, the Box-Muller identity, sample moments, and independence across walkers and steps."""
import math

import numpy as np

from oracle import rng_oracle as rng

# (counter, key) -> output, Philox4x32 with 10 rounds
KAT = [
    ((0x00000000, 0x00000000, 0x00000000, 0x00000000), (0x00000000, 0x00000000),
     (0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8)),
    ((0xffffffff, 0xffffffff, 0xffffffff, 0xffffffff), (0xffffffff, 0xffffffff),
     (0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd)),
    ((0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344), (0xa4093822, 0x299f31d0),          # digits of pi
     (0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1)),
]


def test_known_answer_vectors():
    for ctr, key, out in KAT:
        assert rng.philox4x32_10(ctr, key) == out
        arr = rng.philox4x32_10_array(*[np.array([c]) for c in ctr], key[0], key[1])
        assert tuple(int(a[0]) for a in arr) == out


def test_a_dropped_round_or_a_swapped_multiplier_fails_the_vectors(monkeypatch):
    ctr, key, out = KAT[2]
    monkeypatch.setattr(rng, "M0", rng.M1)
    assert rng.philox4x32_10(ctr, key) != out


def test_uniforms_are_midpoints_of_a_2_to_53_grid_strictly_inside_the_unit_interval():
    lo = np.array([0, 0xFFFFFFFF, 0x800, 0x7FF], dtype=np.uint64)
    hi = np.array([0, 0xFFFFFFFF, 0, 0], dtype=np.uint64)
    u = rng.uniform53(lo, hi)
    assert u[0] == 2.0 ** -54 and u[1] == 1.0 - 2.0 ** -54          # never 0, never 1: log(u1) is finite
    assert u[2] == 1.5 * 2.0 ** -53 and u[3] == u[0]                 # the low 11 bits are dropped


def test_box_muller_identity_and_layout():
    seed, step, nw, ng = 0x123456789ABCDEF, 7, 3, 9                  # odd n_gamma: the last pair is cut
    x = rng.sample_fields(seed, step, nw, ng)
    assert x.shape == (nw, ng) and x.dtype == np.float64
    for w in range(nw):
        for b in range(ng // 2):
            r = rng.philox4x32_10((b, w, step, 0), (seed & 0xFFFFFFFF, seed >> 32))
            u1 = ((((r[1] << 32) | r[0]) >> 11) + 0.5) * 2.0 ** -53
            u2 = ((((r[3] << 32) | r[2]) >> 11) + 0.5) * 2.0 ** -53
            assert abs(x[w, 2 * b] ** 2 + x[w, 2 * b + 1] ** 2 + 2.0 * math.log(u1)) < 1e-12
            assert abs(math.atan2(x[w, 2 * b + 1], x[w, 2 * b]) % (2 * math.pi) - 2 * math.pi * u2) < 1e-9
    assert np.array_equal(rng.sample_fields(seed, step, 1, ng, first_walker=2), x[2:3])       # a walker's fields do not depend on the batch
    assert np.array_equal(rng.sample_fields(seed, step, nw, 4), x[:, :4])


def test_moments_and_independence():
    x = rng.sample_fields(2024, 0, 400, 1000)                        # 4e5 samples
    assert abs(x.mean()) < 5e-3 and abs(x.var() - 1.0) < 1e-2
    assert abs((x ** 4).mean() - 3.0) < 0.05 and abs((x ** 3).mean()) < 0.02
    assert abs(np.mean(x[:, 0::2] * x[:, 1::2])) < 5e-3              # the two outputs of a pair
    assert abs(np.mean(x[:-1] * x[1:])) < 5e-3                       # neighbouring walkers
    y = rng.sample_fields(2024, 1, 400, 1000)                        # next step
    assert abs(np.mean(x * y)) < 5e-3 and not np.array_equal(x, y)
    z = rng.sample_fields(2025, 0, 400, 1000)                        # another seed
    assert abs(np.mean(x * z)) < 5e-3
    assert np.all(np.abs(x) < 10.5)                                  # sqrt(-2 ln 2^-54) = 8.65 is the largest possible radius
