"""Device-resident test integrands (-m gpu): per-sample ln f against the oracle, and
whole AC / AV / portfolio loops running on the device against closed-form integrals."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

FIG6 = dict(centers=[[4.0, 0.0, 0.0], [-4.0, 0.0, 0.0]], sigmas=[math.sqrt(2.0)] * 2, ln_amps=[0.0, 0.0])
LO3, HI3 = np.full(3, -10.0), np.full(3, 10.0)


def _run(kind, f, lo, hi, N, n_iter, **kw):
    from paper_2505_11655_b200 import Ile, Integrator, result_from_device
    ile = Ile(0)
    g = Integrator(ile, kind, len(lo), lo, hi, 2024, N, **kw)
    res = [result_from_device(g.step_integrand(f, N, it))[0] for it in range(n_iter)]
    return ile, g, res


@pytest.mark.parametrize("kind", ["UNIFORM", "AC", "AV", "PORTFOLIO"])
def test_fig6_mixture_parity_and_closed_form(kind):
    from paper_2505_11655_b200 import Integrand
    from oracle.integrands import gaussian_mix_box_integral, ln_gaussian_mix
    from oracle.reduce import reduce_lnw
    f = Integrand.gaussian_mix(**FIG6)
    N = 1 << 17
    kw = dict(N_min_star=2048) if kind in ("AV", "PORTFOLIO") else {}
    ile, g, res = _run(kind, f, LO3, HI3, N, 8, **kw)
    z, lp, lnf, lnw = [t.cpu().numpy() for t in g.last_batch(N)]
    inbox = np.all((z >= LO3[:, None]) & (z < HI3[:, None]), axis=0)
    ref = np.where(inbox, ln_gaussian_mix(z, **FIG6), -np.inf)
    assert np.array_equal(np.isfinite(ref), np.isfinite(lnf))
    np.testing.assert_allclose(lnf[inbox], ref[inbox], rtol=0, atol=1e-12)
    red = reduce_lnw(np.where(inbox, ref - lp, -np.inf))
    assert abs(res[-1]["ln_integral"] - red["ln_integral"]) <= 1e-8
    exact = gaussian_mix_box_integral(LO3, HI3, **FIG6)
    last = res[-1]
    # cumulative estimate over all 8 iterations: unbiased for UNIFORM / AC / PORTFOLIO (their support is
    # the whole box: AC's floor, the portfolio's AC and GMM members); AV misses at most 1 - P_thr
    est, sig = math.exp(last["cum_ln_integral"]), math.exp(last["cum_ln_integral"]) * math.sqrt(max(last["cum_rel_variance"], 0.0))
    lo_f = 0.995 if kind == "AV" else 1.0
    assert lo_f * exact - 5 * sig <= est <= exact + 5 * sig, (est, exact, sig)
    if kind != "UNIFORM":
        assert res[-1]["n_eff"] > 2 * res[0]["n_eff"]                  # adaptation pays (Fig. 3)


def test_rosenbrock_2d_against_quadrature():
    from paper_2505_11655_b200 import Integrand
    from oracle.integrands import ln_rosenbrock
    lo, hi = np.array([-3.0, -2.0]), np.array([3.0, 8.0])
    f = Integrand.rosenbrock(1.0, 100.0, 20.0)
    N = 1 << 17
    ile, g, res = _run("AV", f, lo, hi, N, 8, N_min_star=2048)
    z, lp, lnf, lnw = [t.cpu().numpy() for t in g.last_batch(N)]
    np.testing.assert_allclose(lnf, ln_rosenbrock(z, 1.0, 100.0, 20.0), rtol=0, atol=1e-11)
    x, w = np.polynomial.legendre.leggauss(600)
    xs = 0.5 * (hi[0] - lo[0]) * x + 0.5 * (hi[0] + lo[0])
    ys = 0.5 * (hi[1] - lo[1]) * x + 0.5 * (hi[1] + lo[1])
    X, Y = np.meshgrid(xs, ys, indexing="ij")
    vals = np.exp(ln_rosenbrock(np.stack([X.ravel(), Y.ravel()]), 1.0, 100.0, 20.0)).reshape(600, 600)
    exact = 0.25 * (hi[0] - lo[0]) * (hi[1] - lo[1]) * (w[:, None] * w[None, :] * vals).sum()
    last = res[-1]
    est = math.exp(last["ln_integral"])
    sig = est * math.sqrt(max(last["rel_variance"], 0.0))
    assert 0.99 * exact - 5 * sig <= est <= exact + 5 * sig, (est, exact, sig)
    assert last["n_eff"] / N > 0.02                                     # Fig. 3: AV samples this efficiently


def test_integrand_argument_errors():
    from paper_2505_11655_b200 import Ile, IleError, Integrand, Integrator
    ile = Ile(0)
    g = Integrator(ile, "AC", 1, [0.0], [1.0], 1, 100)
    with pytest.raises(IleError):
        g.step_integrand(Integrand.rosenbrock(), 100, 0)               # d = 1
    f = Integrand.gaussian_mix([[0.5]], [0.1], [0.0])
    f.n_comp = 9
    with pytest.raises(IleError):
        g.step_integrand(f, 100, 0)
