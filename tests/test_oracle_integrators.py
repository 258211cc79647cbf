"""Pins P7, P9, P10, P11 for oracle/reduce.py and oracle/integrators.py: closed-form integrals
and invariants (the paper prints no worked numbers; PAPER.md:261 gives Fig. 6's integrand)."""
import math

import numpy as np
import pytest
from scipy import special, stats

from oracle import integrators as og
from oracle.reduce import combine, reduce_lnw


def gauss_box_integral(mu, sig, lo, hi):
    val = 1.0
    for c in range(len(mu)):
        val *= sig[c] * math.sqrt(2 * math.pi) * 0.5 * (
            special.erf((hi[c] - mu[c]) / (sig[c] * math.sqrt(2))) - special.erf((lo[c] - mu[c]) / (sig[c] * math.sqrt(2))))
    return val


def ln_gauss(z, mu, sig):
    out = np.zeros(z.shape[1])
    for c in range(len(mu)):
        out += -0.5 * ((z[c] - mu[c]) / sig[c]) ** 2
    return out


def run(integ, lnf, N, n_iter, g0=0):
    res = []
    V = None
    for g in range(g0, g0 + n_iter):
        z, ln_ps = integ.draw(N, g)
        lnw = lnf(z) - ln_ps
        lnw = np.where(og.in_box(z, integ.lo, integ.hi), lnw, -np.inf)
        res.append(reduce_lnw(lnw))
        integ.update(z, lnw, ln_ps)
    return res


# ------------------------------------------------------------------------------- qfix
def test_qfix_matches_exp_and_edges():
    t = -np.linspace(0, 29, 5001)
    q = og.qfix(t).astype(np.float64)
    ref = np.exp(t) * 2.0 ** 40
    assert np.all(np.abs(q - ref) <= 0.5 + 4e-16 * ref * 8)
    assert og.qfix(np.array([0.0]))[0] == 1 << 40
    assert og.qfix(np.array([-29.01, -np.inf, np.nan, -1e300])).tolist() == [0, 0, 0, 0]
    assert og.qfix(np.array([-math.log(2.0)]))[0] in ((1 << 39) - 1, 1 << 39, (1 << 39) + 1)


# ------------------------------------------------------------------------------- P7 reductions
def test_reduce_constant_integrand():
    N = 1000
    V0 = 3.5
    r = reduce_lnw(np.full(N, math.log(2.0) + math.log(V0)))      # f = 2, p_s = 1/V0
    assert abs(r["ln_integral"] - math.log(2.0 * V0)) < 1e-15
    assert r["n_eff"] == N and r["n_ess"] == N and abs(r["rel_variance"]) < 1e-18


def test_reduce_hand_example_and_nonfinite():
    w = np.array([1.0, 2.0, 4.0, 0.0, 1.0])
    lnw = np.log(np.where(w > 0, w, 1.0))
    lnw[3] = -np.inf
    r = reduce_lnw(lnw + 700.0)                                    # dynamic-range shift
    assert abs(r["ln_integral"] - (math.log(8.0 / 5.0) + 700.0)) < 1e-12
    assert abs(r["n_eff"] - 8.0 / 4.0) < 1e-12                      # Eq. 9: sum w / max w
    assert abs(r["n_ess"] - 64.0 / 22.0) < 1e-12                    # Eq. 16
    var_w = np.mean(w ** 2) - np.mean(w) ** 2
    assert abs(r["rel_variance"] - var_w / (5 * np.mean(w) ** 2)) < 1e-12
    assert r["n_eff"] <= r["n_ess"] <= 5
    r2 = reduce_lnw(np.array([np.nan, 0.0, np.inf]))
    assert r2["n_nonfinite"] == 2 and r2["n_samples"] == 3
    r3 = reduce_lnw(np.array([-np.inf, -np.inf]))
    assert r3["ln_integral"] == -math.inf and r3["n_eff"] == 0
    # combine == reduce over the union
    a, b = np.array([0.1, 5.0, -3.0]), np.array([7.0, -np.inf])
    c = combine([reduce_lnw(a), reduce_lnw(b)])
    u = reduce_lnw(np.concatenate([a, b]))
    for k in ("ln_integral", "n_eff", "n_ess", "rel_variance"):
        assert abs(c[k] - u[k]) < 1e-13


def test_uniform_mc_gaussian_closed_form_and_variance():
    lo, hi = np.array([-3.0, 0.0, -1.0]), np.array([4.0, 2.0, 5.0])
    mu, sig = [0.5, 1.2, 1.0], [0.8, 0.5, 1.5]
    exact = gauss_box_integral(mu, sig, lo, hi)
    est, sg = [], []
    for seed in range(100):
        r = run(og.Uniform(lo, hi, seed), lambda z: ln_gauss(z, mu, sig), 4096, 1)[0]
        est.append(math.exp(r["ln_integral"]))
        sg.append(math.sqrt(r["rel_variance"]) * est[-1])
    est, sg = np.array(est), np.array(sg)
    assert np.all(np.abs(est - exact) < 4.5 * sg)
    assert 0.7 < est.std() / sg.mean() < 1.3                        # reported variance is the real one
    assert abs(est.mean() - exact) < 4 * sg.mean() / 10


def test_fig6_two_gaussian_integrand():
    # PAPER.md:261 (Fig. 6): two Gaussians, sigma = sqrt(2), centres (+-4, 0, 0)
    lo, hi = np.full(3, -12.0), np.full(3, 12.0)
    s = math.sqrt(2.0)

    def lnf(z):
        a = ln_gauss(z, [4.0, 0, 0], [s] * 3)
        b = ln_gauss(z, [-4.0, 0, 0], [s] * 3)
        return np.logaddexp(a, b)
    exact = gauss_box_integral([4.0, 0, 0], [s] * 3, lo, hi) + gauss_box_integral([-4.0, 0, 0], [s] * 3, lo, hi)
    for kind in ("UNIFORM", "AC", "AV"):
        integ = og.make_integrator(kind, lo, hi, 11, n_bins=30, N_min_star=512)
        res = run(integ, lnf, 1 << 14, 6)
        tot = combine(res[2:])
        sigma = math.sqrt(max(tot["rel_variance"], 1e-12))
        tol = 5 * sigma + (0.002 if kind == "AV" else 0.0)          # AV drops <= 1 - P_thr of the mass
        assert abs(math.exp(tot["ln_integral"]) / exact - 1.0) < tol, kind
        assert tot["n_eff"] <= tot["n_ess"] <= tot["n_samples"]


# ------------------------------------------------------------------------------- P9 AC
def test_ac_invariants_and_adaptation():
    lo, hi = np.array([0.0, -1.0]), np.array([2 * math.pi, 1.0])
    ac = og.AC(lo, hi, 5, n_bins=20, eps=0.1)
    assert np.allclose(ac.pi.sum(axis=1), 1.0)
    # constant integrand: pi stays uniform, estimate exact
    r = run(ac, lambda z: np.zeros(z.shape[1]), 4000, 2)
    assert abs(math.exp(r[1]["ln_integral"]) - og.box_volume(lo, hi)) < 0.05 * og.box_volume(lo, hi)
    assert np.abs(ac.pi - 0.05).max() < 0.02
    # Gaussian: variance falls after adaptation, estimates unbiased, draws land in the drawn bin
    mu, sig = [2.0, 0.3], [0.3, 0.1]
    exact = gauss_box_integral(mu, sig, lo, hi)
    ac = og.AC(lo, hi, 6, n_bins=50, eps=0.1)
    res = run(ac, lambda z: ln_gauss(z, mu, sig), 1 << 14, 6)
    assert res[-1]["rel_variance"] < 0.2 * res[0]["rel_variance"]
    for r in res:
        assert abs(math.exp(r["ln_integral"]) / exact - 1) < 5 * math.sqrt(r["rel_variance"])
    assert np.allclose(ac.pi.sum(axis=1), 1.0, atol=1e-14)
    assert np.allclose(ac.cdf[:, -1], 1.0, atol=1e-13)
    z, ln_ps = ac.draw(5000, 9)
    assert og.in_box(z, lo, hi).all()
    # ln_ps is the product pdf, which integrates to 1: sum_b pi_b = 1 per dimension
    for c in range(2):
        b = og.bin_index(z[c], lo[c], hi[c], 50)
        assert np.all(ac.cdf[c, b] <= ac.cdf[c, b + 1])
    np.testing.assert_allclose(ln_ps, ac.ln_pdf(z))
    # histogram is integer and order independent
    lnw = ln_gauss(z, mu, sig) - ln_ps
    H1 = ac.histogram(z, lnw)
    perm = np.random.default_rng(0).permutation(5000)
    H2 = ac.histogram(z[:, perm], lnw[perm])
    assert H1.dtype == np.uint64 and np.array_equal(H1, H2)
    assert int(H1[0].sum()) == int(H1[1].sum()) == int(og.qfix(lnw - lnw.max()).sum())


def test_ac_draw_inverse_cdf_statistics():
    lo, hi = np.array([0.0]), np.array([1.0])
    ac = og.AC(lo, hi, 8, n_bins=4, eps=0.0)
    ac.pi[0] = [0.1, 0.2, 0.3, 0.4]
    ac._scan()
    z, ln_ps = ac.draw(200000, 0)
    h = np.bincount((z[0] * 4).astype(int), minlength=4) / 200000.0
    assert np.abs(h - ac.pi[0]).max() < 5e-3
    np.testing.assert_allclose(np.exp(ln_ps), ac.pi[0][(z[0] * 4).astype(int)] * 4)


# ------------------------------------------------------------------------------- P10 AV
def test_av_constant_integrand_tie_rule():
    lo, hi = np.zeros(2), np.ones(2)
    av = og.AV(lo, hi, 3, P_thr=0.9, N_min_star=16)
    z, ln_ps = av.draw(1000, 0)
    assert np.all(ln_ps == 0.0) and av.n == 1 and len(av.keys) == 1
    av.update(z, np.zeros(1000))
    # ties: the first N_min by index are kept (G23); N_P = ceil(0.9 * 1000)
    assert av.N_min == 900
    dv = (900 / 1000) / math.sqrt(900)
    n = av.n
    assert n ** 2 <= 1 / dv < (n + 1) ** 2
    assert np.array_equal(av.keys, np.unique(av.key_of(z[:, :900], n)))
    assert len(av.keys) <= av.N_min


def test_av_gaussian_volume_and_estimate():
    d = 3
    lo, hi = np.full(d, -10.0), np.full(d, 10.0)
    sig = [0.7, 1.0, 1.3]
    av = og.AV(lo, hi, 21, P_thr=0.99, N_min_star=256)
    lnf = lambda z: ln_gauss(z, [0.0] * d, sig)
    res = run(av, lnf, 1 << 15, 8)
    exact = gauss_box_integral([0.0] * d, sig, lo, hi)
    # kept volume ~ ellipsoid holding P_thr of the mass: pi^{d/2} r^d prod(sig) / Gamma(d/2+1)
    r2 = stats.chi2.ppf(0.99, d)
    vol = math.pi ** (d / 2) * r2 ** (d / 2) * np.prod(sig) / math.gamma(d / 2 + 1)
    V0 = og.box_volume(lo, hi)
    assert 0.8 * vol < av.v * V0 < 2.5 * vol                 # cells over-cover the ellipsoid a little
    last = res[-1]
    est = math.exp(last["ln_integral"])
    assert est > 0.99 * exact * (1 - 5 * math.sqrt(last["rel_variance"])) - 1e-12
    assert est < exact * (1 + 5 * math.sqrt(last["rel_variance"]))
    assert last["n_ess"] > 0.1 * (1 << 15)                   # high sampling efficiency
    assert len(av.keys) <= av.N_min and av.n <= av.n_max
    # Eq. 13: n^d <= 1/dv < (n+1)^d was enforced with the volume *before* the last update
    assert og.av_n_max(6) ** 6 < 2 ** 62 <= (og.av_n_max(6) + 1) ** 6
    # membership pdf
    z, ln_ps = av.draw(2000, 99)
    np.testing.assert_allclose(av.ln_pdf(z), ln_ps)
    far = np.full((d, 1), 9.5)
    assert av.ln_pdf(far)[0] == -np.inf


def test_av_member_rule_reduces_to_standalone_on_uniform_ps():
    """SURVEY 8(c) "AV as a portfolio member": with the uniform p_s of the AV's own draw the importance
    estimate of the kept volume, (1/(N V0)) sum_kept 1/p_s, is v_g N_min / N, so the
    member rule must leave exactly the state the standalone rule leaves."""
    d = 3
    lo, hi = np.array([-2.0, 0.0, 1.0]), np.array([2.0, 3.0, 6.0])       # V0 = 60: a misplaced V0 cannot hide
    lnf = lambda z: ln_gauss(z, [0.3, 1.2, 3.0], [0.4, 0.5, 0.9])
    a = og.AV(lo, hi, 5, P_thr=0.98, N_min_star=128)
    b = og.AV(lo, hi, 5, P_thr=0.98, N_min_star=128)
    for g in range(4):
        z, ln_ps = a.draw(1 << 13, g)
        zb, ln_psb = b.draw(1 << 13, g)
        assert np.array_equal(z, zb) and np.array_equal(ln_ps, ln_psb)
        lnw = lnf(z) - ln_ps
        a.update(z, lnw, None)                                            # standalone rule
        b.update(z, lnw, ln_ps)                                           # member rule, uniform p_s
        assert (a.n, a.N_min) == (b.n, b.N_min)
        assert abs(b.L_thr - (a.L_thr + ln_ps[0])) < 1e-12                # ln f = ln w + ln p_s: a constant shift here
        assert np.array_equal(a.keys, b.keys)
        assert abs(b.v_new / a.v_new - 1.0) < 1e-14
    assert a.n > 1 and len(a.keys) > 1


def test_av_member_rule_volume_from_nonuniform_samples():
    """Same rule on samples from a known non-uniform density: integrand = indicator of a box B of known
    volume, samples from a product density with hand-set marginals (AC draw, pi set by hand).  With
    P_thr = 1 every sample inside B is kept, and v' V0 = (1/N) sum_{in B} 1/p_s is the unbiased
    importance estimate of vol(B): it must equal vol(B) within Monte Carlo error.  A dropped exp(-mn),
    a V0 on the wrong side or a missing 1/N is off by factors, not per cent."""
    d = 3
    lo, hi = np.array([-1.0, 0.0, 2.0]), np.array([3.0, 2.0, 5.0])       # V0 = 24
    V0 = og.box_volume(lo, hi)
    ac = og.AC(lo, hi, 77, n_bins=8)
    ramp = np.linspace(1.0, 3.0, 8)
    for c in range(d):
        ac.pi[c] = (ramp if c != 1 else ramp[::-1]) / ramp.sum()
    ac._scan()
    N = 1 << 17
    z, ln_ps = ac.draw(N, 0)
    blo, bhi = np.array([0.0, 0.5, 2.5]), np.array([2.0, 1.5, 4.0])      # vol(B) = 2 * 1 * 1.5 = 3
    vol = float(np.prod(bhi - blo))
    inside = og.in_box(z, blo, bhi)
    lnw = np.where(inside, -ln_ps, -np.inf)                               # ln(f p / p_s), f = 1 in B, p = 1
    av = og.AV(lo, hi, 1, P_thr=1.0, N_min_star=1)
    av.update(z, lnw, ln_ps)
    assert av.N_min == int(inside.sum())
    # Monte Carlo error bound: Var(1_B / p_s) <= E[(1_B / p_s)^2] = int_B 1/p_s <= vol(B) max(1/p_s)
    sigma = math.sqrt(vol * math.exp(-ln_ps.min()) / N)
    assert abs(av.v_new * V0 - vol) < 5 * sigma
    assert sigma < 0.03 * vol                                             # ... and the bound is tight enough to matter
    # Eq. 13 with that volume: n^d <= sqrt(N_min) / v' < (n + 1)^d, and the cells cover B, not more than a layer around it
    inv_dv = math.sqrt(av.N_min) / av.v_new
    assert av.n ** d <= inv_dv < (av.n + 1) ** d
    cover = len(av.keys) / float(av.n) ** d * V0
    layer = np.prod(bhi - blo + 2 * (hi - lo) / av.n)
    assert 0.9 * vol < cover <= layer


# ------------------------------------------------------------------------------- GMM + P11 portfolio
def test_gmm_pdf_normalised_and_em_moves_to_target():
    lo, hi = np.array([-8.0, -8.0]), np.array([8.0, 8.0])
    gm = og.GMM(lo, hi, 4, n_comp=3)
    # pdf integrates to ~1 over a wide grid (untruncated mixture; wide box)
    g = np.linspace(-40, 40, 801)
    X, Y = np.meshgrid(g, g, indexing="ij")
    pdf = np.exp(gm.ln_pdf(np.stack([X.ravel(), Y.ravel()]))).reshape(X.shape)
    assert abs(pdf.sum() * 0.1 * 0.1 - 1.0) < 1e-3
    # draws follow the pdf: mean of exp(-ln_ps) over in-box draws ~ box volume fraction
    mu, sig = [2.0, -1.0], [0.5, 0.8]
    res = run(gm, lambda z: ln_gauss(z, mu, sig), 1 << 13, 12)
    exact = gauss_box_integral(mu, sig, lo, hi)
    assert res[-1]["n_ess"] > 5 * res[0]["n_ess"]
    tot = combine(res[6:])
    assert abs(math.exp(tot["ln_integral"]) / exact - 1) < 5 * math.sqrt(tot["rel_variance"]) + 1e-3
    top = np.argmax(gm.omega)
    assert np.abs(gm.mu[top] - mu).max() < 0.2


def test_portfolio_single_member_is_member_and_allocation():
    lo, hi = np.array([-5.0, -5.0]), np.array([5.0, 5.0])
    lnf = lambda z: ln_gauss(z, [1.0, -1.0], [0.4, 0.6])
    for kind in ("AC", "AV"):
        a = og.make_integrator(kind, lo, hi, 17, n_bins=25, N_min_star=128)
        p = og.Portfolio([og.make_integrator(kind, lo, hi, 17, n_bins=25, N_min_star=128)])
        for g in range(3):
            za, la = a.draw(3000, g)
            zp, lp = p.draw(3000, g)
            assert np.array_equal(za, zp) and np.array_equal(la, lp)
            lnw = lnf(za) - la
            a.update(za, lnw, None)
            p.update(zp, lnw, lp)
    # allocation: floor(N W) + remainder in index order; sums to N
    pf = og.make_integrator("PORTFOLIO", lo, hi, 3, members=["AC", "AV", "GMM"], n_gmm=2, N_min_star=64, n_bins=10)
    pf.W = np.array([0.5, 0.3, 0.2])
    Na = pf.allocation(1001)
    assert Na.sum() == 1001 and Na.tolist() == [501, 300, 200]
    res = run(pf, lnf, 6000, 8)
    exact = gauss_box_integral([1.0, -1.0], [0.4, 0.6], lo, hi)
    tot = combine(res[3:])
    assert abs(math.exp(tot["ln_integral"]) / exact - 1) < 5 * math.sqrt(tot["rel_variance"]) + 2e-3
    assert abs(pf.W.sum() - 1) < 1e-14 and pf.W.min() >= 0.05 / 3 / (1 + 0.05) - 1e-12
    # mixture pdf integrates to 1 (d = 2 quadrature over the box; GMM tail outside is small)
    g = np.linspace(-5, 5, 1001)[:-1] + 0.005
    X, Y = np.meshgrid(g, g, indexing="ij")
    pdf = np.exp(pf.ln_pdf(np.stack([X.ravel(), Y.ravel()])))
    gm_in = np.exp(pf.members[2].ln_pdf(np.stack([X.ravel(), Y.ravel()]))).sum() * 1e-4
    want = pf.W[0] + pf.W[1] + pf.W[2] * gm_in
    assert abs(pdf.sum() * 1e-4 - want) < 2e-3


# ------------------------------------------------------------------------------- portfolio options of PAPER.md:297
def _state(m):
    if m.kind == "AC":
        return (m.H.copy(), m.pi.copy())
    if m.kind == "AV":
        return (m.n, m.keys.copy())
    return (m.omega.copy(), m.mu.copy(), m.Sigma.copy())


def test_portfolio_activation_iteration_is_invisible_before_it():
    """A member with first_iter = g0 gets no samples, no density term and no training before g0, and N_s counts the
    activated members only: for g < g0 the portfolio is bit-identical to the portfolio without that member.  At g0
    the weights restart uniform and the newcomer draws its share."""
    lo, hi = np.array([-5.0, -5.0]), np.array([5.0, 5.0])
    lnf = lambda z: ln_gauss(z, [1.0, -1.0], [0.4, 0.6])
    mk = lambda kind, **o: og.make_integrator(kind, lo, hi, 11, **o)
    g0 = 3
    with_late = og.Portfolio([mk("AC", n_bins=10), mk("AV", N_min_star=64), mk("AC", n_bins=30)], first_iter=[0, 0, g0])
    without = og.Portfolio([mk("AC", n_bins=10), mk("AV", N_min_star=64)])
    N = 4000
    for g in range(g0):
        za, la = with_late.draw(N, g)
        zb, lb = without.draw(N, g)
        assert np.array_equal(za, zb) and np.array_equal(la, lb)
        assert with_late.alloc[2] == 0 and with_late.W[2] == 0.0
        lnw = lnf(za) - la
        with_late.update(za, lnw, la)
        without.update(zb, lnw, lb)
        assert np.array_equal(with_late.W[:2], without.W)
        for a in range(2):
            for x, y in zip(_state(with_late.members[a]), _state(without.members[a])):
                assert np.array_equal(x, y)
        assert np.all(with_late.members[2].pi == 1.0 / 30)              # untouched
    z, l = with_late.draw(N, g0)
    assert np.array_equal(with_late.W, np.full(3, 1.0 / 3)) and with_late.alloc.tolist() == [1334, 1333, 1333]
    with_late.update(z, lnf(z) - l, l)
    assert not np.all(with_late.members[2].pi == 1.0 / 30)              # now trained
    with pytest.raises(ValueError):
        og.Portfolio([mk("AC"), mk("AC")], first_iter=[1, 0])


def test_portfolio_silent_member_trains_but_stays_out_of_the_integral():
    """Silent member (listed last): fixed share N // N_active of every batch, no term in p_s, its samples are left
    out of the estimate but train every member (itself included) with the weights L p / p_s."""
    from oracle.ile import iteration
    lo, hi = np.array([-5.0, -5.0]), np.array([5.0, 5.0])
    mu, sig = [1.0, -1.0], [0.4, 0.6]
    pf = og.Portfolio([og.AC(lo, hi, 5, n_bins=20), og.Uniform(lo, hi, 5)], silent=[False, True])
    N = 6000
    z, ln_ps = pf.draw(N, 0)
    assert pf.alloc.tolist() == [3000, 3000] and pf.n_contrib_samples == 3000
    assert np.array_equal(ln_ps, pf.members[0].ln_pdf(z))                # the mixture is the contributing member alone (W = 1)
    lnw = ln_gauss(z, mu, sig) - ln_ps
    ref = og.AC(lo, hi, 5, n_bins=20)
    pf.update(z, lnw, ln_ps)
    assert np.array_equal(pf.members[0].H, ref.histogram(z, lnw))        # trained on all N samples, the silent ones included
    assert pf.members[0].H.sum() > ref.histogram(z[:, :3000], lnw[:3000]).sum()
    assert pf.W.tolist() == [1.0, 0.0]

    class Prob:                                                          # the estimate through oracle.ile.iteration: contributing samples only
        lo_, hi_ = lo, hi
        def lnL_z(self, zz):
            return np.where(og.in_box(zz, lo, hi), ln_gauss(zz, mu, sig), -np.inf)
        def ln_prior(self, zz):
            return np.zeros(zz.shape[1])
    res = []
    for g in range(1, 7):
        out = iteration(Prob(), pf, N, g)
        assert out["result"]["n_samples"] == 3000 and len(out["lnw"]) == N
        res.append(out["result"])
    exact = gauss_box_integral(mu, sig, lo, hi)
    tot = combine(res[2:])
    assert abs(math.exp(tot["ln_integral"]) / exact - 1) < 5 * math.sqrt(tot["rel_variance"]) + 2e-3
    with pytest.raises(ValueError):
        og.Portfolio([og.AC(lo, hi, 5), og.Uniform(lo, hi, 5), og.AC(lo, hi, 5)], silent=[False, True, False])


def test_portfolio_fig7_two_ac_members_second_from_iteration_10():
    """PAPER.md:299 (Fig. 7): a portfolio of two AC integrators with 10 and 30 bins, the high-resolution one joining
    after 10 iterations, on three superposed Gaussians in four dimensions (seeded parameters: the paper's are random
    and unprinted).  The estimate converges to the closed-form integral."""
    d = 4
    lo, hi = np.full(d, -6.0), np.full(d, 6.0)
    rng = np.random.Generator(np.random.Philox(7))
    mus, sigs, amps = rng.uniform(-3, 3, (3, d)), rng.uniform(0.5, 1.0, (3, d)), np.array([1.0, 0.6, 0.3])

    def lnf(z):
        e = np.stack([math.log(amps[c]) + ln_gauss(z, mus[c], sigs[c]) for c in range(3)])
        mx = e.max(axis=0)
        return mx + np.log(np.exp(e - mx).sum(axis=0))
    exact = sum(amps[c] * gauss_box_integral(mus[c], sigs[c], lo, hi) for c in range(3))
    pf = og.make_integrator("PORTFOLIO", lo, hi, 42, members=["AC", "AC"], member_opts=[dict(n_bins=10), dict(n_bins=30)], first_iter=[0, 10])
    res = run(pf, lnf, 1 << 14, 20)
    assert pf.members[0].n_bins == 10 and pf.members[1].n_bins == 30
    assert pf.W[1] > 0.0 and abs(pf.W.sum() - 1) < 1e-14
    tot = combine(res[12:])
    assert abs(math.exp(tot["ln_integral"]) / exact - 1) < 5 * math.sqrt(tot["rel_variance"]) + 2e-3
    assert tot["n_ess"] > 0.05 * 8 * (1 << 14)


# ------------------------------------------------------------------------------- GMM over a subset of dimensions
def test_gmm_dimension_subset():
    """`dims` = the modelled dimensions, the others uniform over the box.  Pins: every dimension listed = the default
    (bit for bit); the density factorises into a lower-dimensional mixture times 1/range and integrates to one;
    draws in the other dimensions are uniform; the EM step moves the modelled marginal onto the target."""
    lo, hi = np.array([-3.0, -8.0, 1.0]), np.array([5.0, 8.0, 4.0])
    full, alld = og.GMM(lo, hi, 9, n_comp=3), og.GMM(lo, hi, 9, n_comp=3, dims=[2, 0, 1])
    za, la = full.draw(2000, 4)
    zb, lb = alld.draw(2000, 4)
    assert np.array_equal(za, zb) and np.array_equal(la, lb)
    # factorisation: a mixture in dimension 1 only == the one-dimensional mixture with the same parameters / (range_0 range_2)
    sub = og.GMM(lo, hi, 9, n_comp=3, dims=[1])
    one = og.GMM(lo[1:2], hi[1:2], 9, n_comp=3)
    one.omega, one.mu, one.Sigma = sub.omega.copy(), sub.mu.copy(), sub.Sigma.copy()
    one._chol()
    z, ln_ps = sub.draw(20000, 0)
    assert np.array_equal(ln_ps, sub.ln_pdf(z))
    np.testing.assert_allclose(ln_ps, one.ln_pdf(z[1:2]) - math.log(8.0 * 3.0), rtol=0, atol=1e-13)
    outside = z.copy()
    outside[0, :5] = 5.5                                                  # outside the box in a uniform dimension: density 0
    assert np.all(sub.ln_pdf(outside)[:5] == -np.inf)
    # the uniform dimensions: inside the box, flat (Kolmogorov-Smirnov), and untouched by the mixture parameters
    for c in (0, 2):
        y = (z[c] - lo[c]) / (hi[c] - lo[c])
        assert y.min() >= 0.0 and y.max() < 1.0 and stats.kstest(y, "uniform").pvalue > 1e-3
    # normalisation by quadrature over (x0 in the box) x (x1 on a wide grid) at fixed x2
    g0 = np.linspace(lo[0], hi[0], 401)[:-1] + (hi[0] - lo[0]) / 800
    g1 = np.linspace(-80.0, 80.0, 8001)[:-1] + 0.01
    X0, X1 = np.meshgrid(g0, g1, indexing="ij")
    pdf = np.exp(sub.ln_pdf(np.stack([X0.ravel(), X1.ravel(), np.full(X0.size, 2.0)])))
    assert abs(pdf.sum() * (hi[0] - lo[0]) / 400 * 0.02 * (hi[2] - lo[2]) - 1.0) < 1e-6
    # EM on a target that is Gaussian in dimension 1 (mean 2.5, sigma 0.7) and flat elsewhere
    for g in range(12):
        z, ln_ps = sub.draw(20000, g + 1)
        lnw = -0.5 * ((z[1] - 2.5) / 0.7) ** 2 - ln_ps
        lnw = np.where(og.in_box(z, lo, hi), lnw, -np.inf)
        sub.update(z, lnw, ln_ps)
    mean = float((sub.omega * sub.mu[:, 0]).sum())
    var = float((sub.omega * (sub.Sigma[:, 0, 0] + (sub.mu[:, 0] - mean) ** 2)).sum())
    assert abs(mean - 2.5) < 0.05 and abs(math.sqrt(var) - 0.7) < 0.08
    assert sub.mu.shape == (3, 1) and sub.Sigma.shape == (3, 1, 1)
