"""Pin P8 (brute-force quadrature over a tiny 2-D extrinsic grid vs Monte Carlo) and the oracle's
integrator loop on the GW likelihood (config 1 shapes)."""
import math

import numpy as np

from oracle import integrators as og
from oracle import likelihood as lk
from oracle.ile import IleProblem, iteration
from oracle.reduce import combine, reduce_lnw
from synth import make_problem


def test_p8_quadrature_vs_mc_two_dims():
    prob = make_problem(1)
    ile = IleProblem(prob)
    th = prob.inj[0]["theta0"]
    fixed = np.array([th["ra"], math.sin(th["dec"]), 0.0, th["phi_ref"], math.cos(th["incl"]), 0.0])
    dims = (2, 5)                                     # psi and distance
    # tensor Gauss-Legendre over (psi, D) of exp(lnL_marg) * p(psi) p(D)
    n = 160
    xg, wg = np.polynomial.legendre.leggauss(n)
    lo, hi = prob.lo[list(dims)], prob.hi[list(dims)]
    a = 0.5 * (hi[0] - lo[0]) * xg + 0.5 * (hi[0] + lo[0])
    b = 0.5 * (hi[1] - lo[1]) * xg + 0.5 * (hi[1] + lo[1])
    A, B = np.meshgrid(a, b, indexing="ij")
    z = np.repeat(fixed[:, None], n * n, axis=1)
    z[2], z[5] = A.ravel(), B.ravel()
    lnL = ile.lnL_z(z)
    lnp = -math.log(math.pi) + np.log(3 * z[5] ** 2 / (prob.D_max ** 3 - prob.D_min ** 3))
    W = (0.5 * (hi[0] - lo[0]) * wg)[:, None] * (0.5 * (hi[1] - lo[1]) * wg)[None, :]
    e = lnL + lnp + np.log(W.ravel())
    ln_quad = e.max() + math.log(np.exp(e - e.max()).sum())
    # Monte Carlo in the same two dimensions (oracle Uniform integrator + Eq. 8)
    parts = []
    for seed in range(4):
        u = og.Uniform(lo, hi, 100 + seed)
        z2, ln_ps = u.draw(1 << 14, 0)
        zz = np.repeat(fixed[:, None], z2.shape[1], axis=1)
        zz[2], zz[5] = z2[0], z2[1]
        lw = ile.lnL_z(zz) - math.log(math.pi) + np.log(3 * zz[5] ** 2 / (prob.D_max ** 3 - prob.D_min ** 3)) - ln_ps
        parts.append(reduce_lnw(lw))
    tot = combine(parts)
    sigma = math.sqrt(tot["rel_variance"])
    assert abs(tot["ln_integral"] - ln_quad) < 4 * sigma + 1e-6, (tot["ln_integral"], ln_quad, sigma)


def test_oracle_ile_loop_config1_small():
    prob = make_problem(1)
    ile = IleProblem(prob)
    res = []
    for seed in (1, 2):
        integ = og.make_integrator("AC", prob.lo, prob.hi, seed, n_bins=50)
        out = [iteration(ile, integ, 1 << 15, g)["result"] for g in range(8)]
        assert all(np.isfinite(o["ln_integral"]) for o in out)
        res.append(combine(out[4:]))
    # two seeds estimate the same evidence (6-D, SNR 10: heavy-tailed weights, loose bound)
    assert abs(res[0]["ln_integral"] - res[1]["ln_integral"]) < 1.5
    # below the Cauchy-Schwarz-like ceiling max lnL and far above the noise-only level
    assert 25.0 < res[0]["ln_integral"] < 0.5 * prob.rho2 + 30.0
    # out-of-box samples get zero weight
    z = np.array([[1.0], [0.2], [0.3], [7.0], [0.1], [300.0]])       # phi_ref = 7 > 2 pi
    assert ile.lnL_z(z)[0] == -np.inf
