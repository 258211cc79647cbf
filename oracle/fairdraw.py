"""Oracle: fair draws from weighted Monte Carlo samples (TEST INFRASTRUCTURE ONLY).

PAPER.md:51 ("fairly drawing some (fixed) number of extrinsic parameters from the underlying ILE
Monte Carlo integral weighted samples"), PAPER.md:115 ("we make a fair draw from these weighted
samples"), PAPER.md:121 (each worker draws a constant multiple of n_eff samples).  The paper does
not name the resampling scheme; reading G39: draws with replacement,
probability of sample i = w_i / sum w, realised either as systematic resampling (one uniform,
M equally spaced positions: every count is within 1 of M w_i / sum w) or as M independent draws.

Bit-exact by construction: weights are the fixed-point q_i = qfix(ln w_i - max) of the integrators
(uint64, 2^40 scale), prefix sums are exact integers, positions use only IEEE * / floor.
"""
from __future__ import annotations

import numpy as np

from .integrators import qfix
from .philox import uniforms


def fair_draw(lnw, M, seed, g, mode="systematic"):
    """Indices [M] (int64) of the drawn samples; -1 everywhere when no sample has positive weight.

    systematic : u0 = uniform 0 of counter (0, g); position j = (j + u0) / M
    independent: u_j = uniform 0 of counter (j, g); position j = u_j
    r_j = floor(position * float(T)) (clamped to T - 1), T = sum q; index = first i with S_i > r_j,
    S the inclusive prefix sums of q."""
    lnw = np.asarray(lnw, dtype=np.float64)
    fin = np.isfinite(lnw)
    out = np.full(M, -1, dtype=np.int64)
    if not fin.any():
        return out
    m = lnw[fin].max()
    q = qfix(np.where(fin, lnw, -np.inf) - m)
    S = np.cumsum(q, dtype=np.uint64)
    T = int(S[-1])
    if T == 0:
        return out
    j = np.arange(M, dtype=np.uint64)
    if mode == "systematic":
        u0 = uniforms(seed, np.zeros(1, dtype=np.uint64), g, 1)[0, 0]
        pos = (j.astype(np.float64) + u0) / float(M)
    else:
        pos = uniforms(seed, j, g, 1)[0]
    r = np.floor(pos * float(T))
    r = np.minimum(r.astype(np.uint64), np.uint64(T - 1))
    return np.searchsorted(S, r, side="right").astype(np.int64)
