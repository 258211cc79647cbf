"""Oracle: Philox4x32-10 counter-based generator (TEST INFRASTRUCTURE ONLY).

The paper is silent on the random-number generator; north_star asks
for a counter-based RNG.  This is the published Philox4x32 round function (Salmon et al.
2011, "Parallel random numbers: as easy as 1, 2, 3") applied 10 times, restated in numpy
integer arithmetic.  Pinned in tests/test_oracle_philox.py against cuRAND's host generator
(a library routine) and by uniformity tests.

Counter layout used by every integrator ("Determinism"):
    counter = (i_lo, i_hi, g, s)  sample index i (64 bit), iteration g, stream s
    key     = (seed_lo, seed_hi)
    uniform e (e = 0, 1, 2, ...) of sample i at iteration g = slot e % 2 of stream s = e // 2
    u = ((hi << 32 | lo) >> 11) * 2^-53, (lo, hi) = words (0, 1) for slot 0, (2, 3) for slot 1
"""
from __future__ import annotations

import numpy as np

_M0 = np.uint64(0xD2511F53)
_M1 = np.uint64(0xCD9E8D57)
_W0 = 0x9E3779B9
_W1 = 0xBB67AE85
_MASK = np.uint64(0xFFFFFFFF)
_SH32 = np.uint64(32)


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    """Ten Philox4x32 rounds.  c0..c3: uint32-valued arrays (any integer dtype); k0, k1 python
    ints.  Returns four uint64 arrays holding 32-bit words."""
    c0 = np.asarray(c0).astype(np.uint64) & _MASK
    c1 = np.asarray(c1).astype(np.uint64) & _MASK
    c2 = np.asarray(c2).astype(np.uint64) & _MASK
    c3 = np.asarray(c3).astype(np.uint64) & _MASK
    k0 = int(k0) & 0xFFFFFFFF
    k1 = int(k1) & 0xFFFFFFFF
    for _ in range(10):
        p0 = _M0 * c0                      # 32x32 -> 64 bit products, exact in uint64
        p1 = _M1 * c2
        hi0, lo0 = p0 >> _SH32, p0 & _MASK
        hi1, lo1 = p1 >> _SH32, p1 & _MASK
        c0, c1, c2, c3 = (hi1 ^ c1 ^ np.uint64(k0)), lo1, (hi0 ^ c3 ^ np.uint64(k1)), lo0
        k0 = (k0 + _W0) & 0xFFFFFFFF
        k1 = (k1 + _W1) & 0xFFFFFFFF
    return c0, c1, c2, c3


def uniforms(seed, i, g, n_uniform):
    """u[e, :] for e = 0..n_uniform-1: uniform doubles in [0,1) for sample indices i (array of
    non-negative ints) at iteration g."""
    i = np.asarray(i, dtype=np.uint64)
    seed = int(seed) & 0xFFFFFFFFFFFFFFFF
    k0, k1 = seed & 0xFFFFFFFF, seed >> 32
    i_lo, i_hi = i & _MASK, i >> _SH32
    out = np.empty((n_uniform, i.shape[0]))
    gs = np.full(i.shape, int(g) & 0xFFFFFFFF, dtype=np.uint64)
    for s in range((n_uniform + 1) // 2):
        r0, r1, r2, r3 = philox4x32_10(i_lo, i_hi, gs, np.full(i.shape, s, dtype=np.uint64), k0, k1)
        u_a = (((r1 << _SH32) | r0) >> np.uint64(11)).astype(np.float64) * 2.0 ** -53
        u_b = (((r3 << _SH32) | r2) >> np.uint64(11)).astype(np.float64) * 2.0 ** -53
        out[2 * s] = u_a
        if 2 * s + 1 < n_uniform:
            out[2 * s + 1] = u_b
    return out
