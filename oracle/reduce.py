"""Oracle: Monte Carlo weight reductions (TEST INFRASTRUCTURE ONLY).

PAPER.md:102-105 Eq. (8) integral estimate; Eq. (9) n_eff = sum p_k / max p_k;
PAPER.md:274-279 Eq. (14)-(16) weights relative to the maximum and n_ESS = (sum w)^2 / sum w^2.
Readings G15 (population variance), G16 (both effective-sample measures returned).
"""
from __future__ import annotations

import math

import numpy as np


def reduce_lnw(lnw):
    """ln w_i = ln L_i + ln p_i - ln p_s,i for one batch of N samples -> dict with
    ln_integral, rel_variance, n_eff, n_ess, ln_w_max, n_samples, n_nonfinite and the raw sums
    S1 = sum exp(ln w - m), S2 = sum exp(2 (ln w - m)).

    Samples with ln w = -inf (zero weight, e.g. outside the box) count in N and contribute 0.
    NaN / +inf are counted in n_nonfinite and contribute 0."""
    lnw = np.asarray(lnw, dtype=np.float64)
    N = lnw.shape[0]
    bad = np.isnan(lnw) | (lnw == np.inf)
    good = ~bad & (lnw > -np.inf)
    out = dict(n_samples=N, n_nonfinite=int(bad.sum()))
    if not good.any():
        out.update(ln_integral=-math.inf, rel_variance=math.inf, n_eff=0.0, n_ess=0.0,
                   ln_w_max=-math.inf, S1=0.0, S2=0.0)
        return out
    m = lnw[good].max()
    e = np.exp(lnw[good] - m)
    S1 = float(e.sum())
    S2 = float((e * e).sum())
    out.update(ln_integral=m + math.log(S1) - math.log(N), n_eff=S1, n_ess=S1 * S1 / S2,
               rel_variance=S2 / (S1 * S1) - 1.0 / N, ln_w_max=float(m), S1=S1, S2=S2)
    return out


def combine(parts):
    """Cumulative estimate over several batches, each sample keeping the p_s it was drawn
    from: the same formulas over the union of all samples."""
    parts = [p for p in parts]
    N = sum(p["n_samples"] for p in parts)
    fin = [p for p in parts if p["S1"] > 0.0]
    if not fin:
        return dict(ln_integral=-math.inf, n_eff=0.0, n_ess=0.0, rel_variance=math.inf,
                    ln_w_max=-math.inf, n_samples=N, S1=0.0, S2=0.0)
    m = max(p["ln_w_max"] for p in fin)
    S1 = sum(p["S1"] * math.exp(p["ln_w_max"] - m) for p in fin)
    S2 = sum(p["S2"] * math.exp(2.0 * (p["ln_w_max"] - m)) for p in fin)
    return dict(ln_integral=m + math.log(S1) - math.log(N), n_eff=S1, n_ess=S1 * S1 / S2,
                rel_variance=S2 / (S1 * S1) - 1.0 / N, ln_w_max=m, n_samples=N, S1=S1, S2=S2)
