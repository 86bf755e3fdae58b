"""CPU ORACLE for the auxiliary-field sampler of the propagation step (Eq. 4: "p(x) is the normal
distribution"; PAPER.md:96-123 draw x once per walker and step).

TEST INFRASTRUCTURE ONLY, like ``afqmc_oracle.py``: only ``tests/`` and the CPU-baseline legs of ``bench.py`` may import
it; it shares no code with ``paper_2209_04015_b200/``.

The paper does not name a generator.  The reading taken here (row 21): a counter-based generator, so
that the CUDA path and this oracle can each implement it and produce the same numbers without passing state around --
Philox4x32-10 (Salmon, Moraes, Dror, Shaw: "Parallel random numbers: as easy as 1, 2, 3", SC'11), restated from the
published algorithm:

    key     = (seed low 32 bits, seed high 32 bits)
    counter = (pair index b = gamma // 2, walker w, step low 32 bits, step high 32 bits)
    (r0, r1, r2, r3) = Philox4x32-10(counter, key)
    u1 = (((r1 << 32 | r0) >> 11) + 0.5) 2^-53,   u2 = (((r3 << 32 | r2) >> 11) + 0.5) 2^-53      both in (0, 1)
    x[w][2b]     = sqrt(-2 ln u1) cos(2 pi u2)                                                      Box-Muller
    x[w][2b + 1] = sqrt(-2 ln u1) sin(2 pi u2)

Pins (tests/test_rng_pins.py): the three known-answer vectors published with the algorithm, the range and resolution of
the uniforms, the Box-Muller identity x0^2 + x1^2 = -2 ln u1, sample moments, and independence across walkers / steps.
"""
from __future__ import annotations

import math

import numpy as np

M0, M1 = 0xD2511F53, 0xCD9E8D57          # round multipliers
W0, W1 = 0x9E3779B9, 0xBB67AE85          # key increments (golden ratio, sqrt(3) - 1)
MASK = 0xFFFFFFFF


def philox4x32_10(counter, key):
    """One block of Philox4x32 with 10 rounds on Python integers: counter = 4 words, key = 2 words -> 4 words."""
    c0, c1, c2, c3 = (int(v) & MASK for v in counter)
    k0, k1 = (int(v) & MASK for v in key)
    for rnd in range(10):
        if rnd:
            k0, k1 = (k0 + W0) & MASK, (k1 + W1) & MASK
        p0, p1 = M0 * c0, M1 * c2                      # 64-bit products
        c0, c1, c2, c3 = ((p1 >> 32) ^ c1 ^ k0) & MASK, p1 & MASK, ((p0 >> 32) ^ c3 ^ k1) & MASK, p0 & MASK
    return c0, c1, c2, c3


def philox4x32_10_array(c0, c1, c2, c3, k0, k1):
    """The same on numpy uint64 arrays holding 32-bit words (broadcast together); returns four uint64 arrays."""
    c0, c1, c2, c3 = (np.asarray(v, dtype=np.uint64) & np.uint64(MASK) for v in np.broadcast_arrays(c0, c1, c2, c3))
    k0, k1 = np.uint64(int(k0) & MASK), np.uint64(int(k1) & MASK)
    m = np.uint64(MASK)
    s32 = np.uint64(32)
    for rnd in range(10):
        if rnd:
            k0, k1 = (k0 + np.uint64(W0)) & m, (k1 + np.uint64(W1)) & m
        p0, p1 = np.uint64(M0) * c0, np.uint64(M1) * c2
        c0, c1, c2, c3 = ((p1 >> s32) ^ c1 ^ k0) & m, p1 & m, ((p0 >> s32) ^ c3 ^ k1) & m, p0 & m
    return c0, c1, c2, c3


def uniform53(lo, hi):
    """(((hi << 32 | lo) >> 11) + 0.5) 2^-53: a uniform in (0, 1) on a grid of 2^53 midpoints, never 0 or 1."""
    word = (np.asarray(hi, dtype=np.uint64) << np.uint64(32)) | np.asarray(lo, dtype=np.uint64)
    return ((word >> np.uint64(11)).astype(np.float64) + 0.5) * 2.0 ** -53


def sample_fields(seed: int, step: int, n_walkers: int, n_gamma: int, first_walker: int = 0) -> np.ndarray:
    """x[w][gamma], float64 [n_walkers][n_gamma], standard normal, for walkers first_walker .. first_walker + n_walkers - 1
    of propagation step `step` under `seed` (header)."""
    nb = (n_gamma + 1) // 2
    b = np.arange(nb, dtype=np.uint64)[None, :]
    w = (np.arange(n_walkers, dtype=np.uint64) + np.uint64(first_walker))[:, None]
    r0, r1, r2, r3 = philox4x32_10_array(b, w, np.uint64(step & MASK), np.uint64((step >> 32) & MASK), seed & MASK, (seed >> 32) & MASK)
    u1, u2 = uniform53(r0, r1), uniform53(r2, r3)
    rad = np.sqrt(-2.0 * np.log(u1))
    out = np.empty((n_walkers, 2 * nb), dtype=np.float64)
    out[:, 0::2] = rad * np.cos(2.0 * math.pi * u2)
    out[:, 1::2] = rad * np.sin(2.0 * math.pi * u2)
    return np.ascontiguousarray(out[:, :n_gamma])
