"""Oracle: one integrator iteration of the ILE loop (TEST INFRASTRUCTURE ONLY).

draw -> evaluate lnL -> ln w = lnL + ln p - ln p_s -> reduce (Eq. 8, 9, 16) -> update sampler
(call stack (2) of SURVEY.md section 3).
"""
from __future__ import annotations

import numpy as np

from . import likelihood as lk
from .reduce import reduce_lnw


class IleProblem:
    """Bundle of the arrays one intrinsic point needs (duck-typed from synth.Problem)."""

    def __init__(self, prob, p=0):
        self.a = dict(D=prob.D, pos=prob.pos, gmst=prob.gmst, ell=prob.ell, m=prob.m,
                      Q=prob.Q[p], U=prob.U[p], V=prob.V[p], D_ref=prob.D_ref, fs=prob.fs,
                      t_Q0=prob.t_Q0, t_lo=prob.t_lo, dt=prob.dt, N_t=prob.N_t)
        self.interp = prob.interp
        self.table = prob.table
        self.D_min, self.D_max = prob.D_min, prob.D_max
        self.lo, self.hi = prob.lo, prob.hi

    def lnL_z(self, z):
        """lnL for in-box samples; -inf outside the box (integrand zero there)."""
        z = np.asarray(z, dtype=np.float64)
        ok = np.ones(z.shape[1], dtype=bool)
        for c in range(z.shape[0]):
            ok &= (z[c] >= self.lo[c]) & (z[c] < self.hi[c])
        out = np.full(z.shape[1], -np.inf)
        if ok.any():
            out[ok] = lk.lnL_z(z=z[:, ok], interp=self.interp, table=self.table, **self.a)
        return out

    def ln_prior(self, z):
        return lk.ln_prior_z(np.asarray(z), self.D_min, self.D_max)


def iteration(ile, integ, N, g, update=True):
    """One pass: returns dict(z, ln_ps, lnL, lnw, result)."""
    z, ln_ps = integ.draw(N, g)
    lnL = ile.lnL_z(z)
    with np.errstate(invalid="ignore"):
        lnw = lnL + ile.ln_prior(z) - ln_ps
    lnw = np.where(np.isfinite(lnL), lnw, -np.inf)
    # a portfolio's silent members draw after the contributing ones and stay out of the estimate
    res = reduce_lnw(lnw[:getattr(integ, "n_contrib_samples", N)])
    if update:
        # a standalone AV samples uniformly inside its cells, so it follows PAPER.md:265 exactly
        # (V_{g+1} = V_g N_min / N_live); ln p_s matters only to a portfolio member
        integ.update(z, lnw, None if integ.kind == "AV" else ln_ps)
    return dict(z=z, ln_ps=ln_ps, lnL=lnL, lnw=lnw, result=res)
