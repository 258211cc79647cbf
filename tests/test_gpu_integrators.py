"""GPU parity of the integrator kernels (through the C ABI) against the oracle (-m gpu).

Teacher-forced per iteration (SURVEY 8(c) "Determinism"): same state in -> same draws (bit-exact
for UNIFORM / AC / AV) -> the oracle's ln w into both updates -> identical integer state out
(AC histograms, AV n_bins / N_min / sorted key set, portfolio allocations).  GMM parameters and
all densities are floating point: compared to 1e-10 relative.
"""
import math

import numpy as np
import pytest

from synth import make_problem

pytestmark = pytest.mark.gpu

LO6 = np.array([0.0, -1.0, 0.0, 0.0, -1.0, 100.0])
HI6 = np.array([2 * math.pi, 1.0, math.pi, 2 * math.pi, 1.0, 2000.0])


@pytest.fixture(scope="module")
def env():
    import torch
    from paper_2505_11655_b200 import Ile
    prob = make_problem(1)
    ile = Ile(0)
    ile.load_problem(prob)
    return torch, ile, prob


def _dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _gauss_lnw(z, lo, hi, centre=0.35, width=0.07, offset=37.0):
    """Toy integrand: separable Gaussian in unit-cube coordinates (host numpy, not the oracle)."""
    y = (z - lo[:, None]) / (hi - lo)[:, None]
    return offset - 0.5 * (((y - centre) / width) ** 2).sum(axis=0)


def _make(ile, kind, d, N, seed=1234, **kw):
    from paper_2505_11655_b200 import Integrator
    return Integrator(ile, kind, d, LO6[:d], HI6[:d], seed, N, **kw)


def _oracle(kind, d, seed=1234, **kw):
    from oracle.integrators import make_integrator
    return make_integrator(kind, LO6[:d], HI6[:d], seed, **kw)


def test_uniform_draw_bit_exact(env):
    torch, ile, _ = env
    N, d = 100003, 6
    g = _make(ile, "UNIFORM", d, N)
    o = _oracle("UNIFORM", d)
    for it in (0, 7):
        z, lp = g.draw(N, it)
        zo, lpo = o.draw(N, it)
        assert np.array_equal(z.cpu().numpy(), zo)                 # Philox + draw arithmetic: bit-exact
        np.testing.assert_allclose(lp.cpu().numpy(), lpo, rtol=1e-14)


@pytest.mark.parametrize("d,N", [(6, 50021), (3, 4096)])
def test_ac_teacher_forced(env, d, N):
    torch, ile, _ = env
    g = _make(ile, "AC", d, N, n_bins=100, eps=0.1, beta=1.0)
    o = _oracle("AC", d, n_bins=100, eps=0.1, beta=1.0)
    lo, hi = LO6[:d], HI6[:d]
    for it in range(4):
        z, lp = g.draw(N, it)
        zo, lpo = o.draw(N, it)
        zg = z.cpu().numpy()
        assert np.array_equal(zg, zo), f"iteration {it}: draws differ"
        np.testing.assert_allclose(lp.cpu().numpy(), lpo, rtol=0, atol=1e-12)
        lnw = _gauss_lnw(zo, lo, hi) - lpo
        if it == 2:
            lnw[:5] = [np.nan, np.inf, -np.inf, 0.0, -1e9]
        o.update(zo, lnw, lpo)
        g.update(z, _dev(torch, lnw), lp)
        st = g.get_state()
        assert np.array_equal(st["H"], o.H), f"iteration {it}: histograms differ"
        assert np.array_equal(st["pi"], o.pi) and np.array_equal(st["cdf"], o.cdf)
    zt = np.stack([np.random.default_rng(1).uniform(lo[c] - 0.1, hi[c] + 0.1, 999) for c in range(d)])
    np.testing.assert_allclose(g.ln_pdf(_dev(torch, zt)).cpu().numpy(), o.ln_pdf(zt), rtol=0, atol=1e-12)


def test_ac_no_finite_weight_keeps_state(env):
    torch, ile, _ = env
    N, d = 1000, 2
    g = _make(ile, "AC", d, N)
    z, lp = g.draw(N, 0)
    before = g.get_state()
    g.update(z, _dev(torch, np.full(N, -np.inf)), lp)
    after = g.get_state()
    assert np.array_equal(before["pi"], after["pi"]) and not after["H"].any()


@pytest.mark.parametrize("d,N,star", [(6, 65536 + 77, 4096), (2, 20000, 512)])
def test_av_teacher_forced(env, d, N, star):
    torch, ile, _ = env
    g = _make(ile, "AV", d, N, P_thr=0.999, N_min_star=star)
    o = _oracle("AV", d, P_thr=0.999, N_min_star=star)
    lo, hi = LO6[:d], HI6[:d]
    for it in range(6):
        z, lp = g.draw(N, it)
        zo, lpo = o.draw(N, it)
        assert np.array_equal(z.cpu().numpy(), zo), f"iteration {it}: draws differ"
        np.testing.assert_allclose(lp.cpu().numpy(), lpo, rtol=1e-14)
        lnw = _gauss_lnw(zo, lo, hi, width=0.05) - lpo
        if it == 1:
            lnw[3] = np.nan
            lnw[4] = -np.inf
        o.update(zo, lnw, None)
        g.update(z, _dev(torch, lnw), None)
        st = g.get_state()
        assert (st["n"], st["N_min"]) == (o.n, o.N_min), f"iteration {it}: n_bins / N_min differ"
        assert np.array_equal(st["keys"], o.keys), f"iteration {it}: cell sets differ"
        assert st["L_thr"] == o.L_thr
    assert o.n > 1 and len(o.keys) > 1
    zt = np.stack([np.random.default_rng(2).uniform(lo[c], hi[c], 2999) for c in range(d)])
    np.testing.assert_allclose(g.ln_pdf(_dev(torch, zt)).cpu().numpy(), o.ln_pdf(zt), rtol=1e-14)


def test_av_constant_integrand_tie_rule(env):
    """Reading G23: ties are ordered by sample index; a constant integrand keeps the first N_min."""
    torch, ile, _ = env
    N, d = 30000, 3
    g = _make(ile, "AV", d, N, P_thr=0.5, N_min_star=100)
    o = _oracle("AV", d, P_thr=0.5, N_min_star=100)
    for it in range(3):
        z, lp = g.draw(N, it)
        zo, lpo = o.draw(N, it)
        assert np.array_equal(z.cpu().numpy(), zo)
        lnw = np.full(N, 2.5)
        o.update(zo, lnw, None)
        g.update(z, _dev(torch, lnw), None)
        st = g.get_state()
        assert (st["n"], st["N_min"]) == (o.n, o.N_min)
        assert np.array_equal(st["keys"], o.keys)
    assert o.N_min == N // 2


def test_av_member_update_with_nonuniform_ps(env):
    """AV trained on samples from another density (its portfolio role): importance volume."""
    torch, ile, _ = env
    N, d = 40000, 3
    g = _make(ile, "AV", d, N, N_min_star=256)
    o = _oracle("AV", d, N_min_star=256)
    ac = _oracle("AC", d)
    lo, hi = LO6[:d], HI6[:d]
    for it in range(3):
        z, lp = ac.draw(N, it)
        lnw = _gauss_lnw(z, lo, hi) - lp
        ac.update(z, lnw, lp)
        o.update(z, lnw, lp)
        g.update(_dev(torch, z), _dev(torch, lnw), _dev(torch, lp))
        st = g.get_state()
        assert (st["n"], st["N_min"]) == (o.n, o.N_min)
        assert np.array_equal(st["keys"], o.keys)


# (5, 8): config 5's member; (6, 16): the most moments per component the tests' box allows (448 sums: every thread of the EM
# kernel carries two); (2, 3): 18 sums, fourteen slices of a round per sum
@pytest.mark.parametrize("d,n_gmm,N", [(5, 8, 30011), (6, 16, 20003), (2, 3, 7001)])
def test_gmm_parity(env, d, n_gmm, N):
    torch, ile, _ = env
    g = _make(ile, "GMM", d, N, n_gmm=n_gmm)
    o = _oracle("GMM", d, n_gmm=n_gmm)
    lo, hi = LO6[:d], HI6[:d]
    st = g.get_state()
    assert np.array_equal(st["mu"], o.mu) and np.array_equal(st["L"], o.L)      # seeded initial state
    for it in range(3):
        z, lp = g.draw(N, it)
        zo, lpo = o.draw(N, it)
        zg = z.cpu().numpy()
        np.testing.assert_allclose(zg, zo, rtol=0, atol=1e-10 * np.abs(hi - lo).max())
        np.testing.assert_allclose(lp.cpu().numpy(), o.ln_pdf(zg), rtol=0, atol=1e-10)
        lnw = _gauss_lnw(zg, lo, hi, width=0.1) - o.ln_pdf(zg)
        o.update(zg, lnw)
        g.update(z, _dev(torch, lnw))
        st = g.get_state()
        for k, ref in (("omega", o.omega), ("mu", o.mu), ("Sigma", o.Sigma), ("L", o.L)):
            np.testing.assert_allclose(st[k], ref, rtol=1e-10, atol=1e-10 * np.abs(ref).max(), err_msg=f"iteration {it}: {k}")


def test_gmm_dimension_subset_parity(env):
    """gmm_dims_mask: the mixture models dimensions {1, 3} of five, the others are uniform over the box."""
    torch, ile, _ = env
    N, d, dims = 30011, 5, [1, 3]
    g = _make(ile, "GMM", d, N, n_gmm=4, gmm_dims=dims)
    o = _oracle("GMM", d, n_gmm=4, gmm_dims=dims)
    lo, hi = LO6[:d], HI6[:d]
    st = g.get_state()
    assert st["gd"] == 2 and st["mu"].shape == (4, 2)
    assert np.array_equal(st["mu"], o.mu) and np.array_equal(st["L"], o.L)      # seeded initial state
    for it in range(3):
        z, lp = g.draw(N, it)
        zo, lpo = o.draw(N, it)
        zg = z.cpu().numpy()
        np.testing.assert_allclose(zg[dims], zo[dims], rtol=0, atol=1e-10 * np.abs(hi - lo).max())
        assert np.array_equal(zg[[0, 2, 4]], zo[[0, 2, 4]])                     # the uniform dimensions: bit-exact
        ref = o.ln_pdf(zg)
        assert np.array_equal(np.isfinite(ref), np.isfinite(lp.cpu().numpy()))
        np.testing.assert_allclose(lp.cpu().numpy(), ref, rtol=0, atol=1e-10)
        out = zg.copy()
        out[0, :7] = hi[0] + 1.0                                               # outside the box in a uniform dimension: density 0
        assert np.all(g.ln_pdf(_dev(torch, out)).cpu().numpy()[:7] == -np.inf)
        lnw = _gauss_lnw(zg, lo, hi, width=0.1) - ref
        o.update(zg, lnw)
        g.update(z, _dev(torch, lnw))
        st = g.get_state()
        for k, r in (("omega", o.omega), ("mu", o.mu), ("Sigma", o.Sigma), ("L", o.L)):
            np.testing.assert_allclose(st[k], r, rtol=1e-10, atol=1e-10 * np.abs(r).max(), err_msg=f"iteration {it}: {k}")
    with pytest.raises(Exception):
        _make(ile, "GMM", 3, 100, gmm_dims=[4])                                # a dimension >= d


def _load_portfolio_state(o, st):
    """Copy a parsed GPU state into the oracle portfolio (teacher forcing: same state in)."""
    o.W = st["W"][:o.Ns].copy()
    o.frozen = st["frozen"][:o.Ns].astype(bool)
    for mem, ms in zip(o.members, st["members"]):
        if mem.kind == "AC":
            mem.H, mem.pi, mem.cdf = ms["H"].copy(), ms["pi"].copy(), ms["cdf"].copy()
        elif mem.kind == "AV":
            mem.n, mem.keys, mem.N_min, mem.L_thr = ms["n"], ms["keys"].copy(), ms["N_min"], ms["L_thr"]
        elif mem.kind == "GMM":
            mem.omega, mem.mu, mem.Sigma, mem.L = ms["omega"].copy(), ms["mu"].copy(), ms["Sigma"].copy(), ms["L"].copy()


def test_portfolio_teacher_forced(env):
    torch, ile, _ = env
    N, d = 60000, 4
    kw = dict(n_bins=50, eps=0.1, beta=1.0, P_thr=0.999, N_min_star=1024, n_gmm=4)
    g = _make(ile, "PORTFOLIO", d, N, members=("AC", "AV", "GMM"), **kw)
    o = _oracle("PORTFOLIO", d, members=["AC", "AV", "GMM"], **kw)
    lo, hi = LO6[:d], HI6[:d]
    for it in range(4):
        _load_portfolio_state(o, g.get_state())
        z, lp = g.draw(N, it)
        zo, lpo = o.draw(N, it)
        zg = z.cpu().numpy()
        st = g.get_state()
        assert np.array_equal(st["alloc"][:3], o.alloc), f"iteration {it}: allocations differ"
        na, nv = int(o.alloc[0]), int(o.alloc[1])
        assert np.array_equal(zg[:, :na + nv], zo[:, :na + nv])               # AC and AV segments bit-exact
        np.testing.assert_allclose(zg[:, na + nv:], zo[:, na + nv:], rtol=0, atol=1e-9)
        lpg = lp.cpu().numpy()
        ref = o.ln_pdf(zg)
        assert np.array_equal(np.isfinite(lpg), np.isfinite(ref))
        fin = np.isfinite(ref)
        np.testing.assert_allclose(lpg[fin], ref[fin], rtol=0, atol=1e-10)
        lnw = np.where(fin, _gauss_lnw(zg, lo, hi, width=0.08) - ref, -np.inf)
        inbox = np.all((zg >= lo[:, None]) & (zg < hi[:, None]), axis=0)
        lnw = np.where(inbox, lnw, -np.inf)
        o.alloc = st["alloc"][:3].copy()
        o.update(zg, lnw, ref)
        g.update(z, _dev(torch, lnw), _dev(torch, ref))
        st = g.get_state()
        np.testing.assert_allclose(st["W"][:3], o.W, rtol=1e-11)
        assert np.array_equal(st["frozen"][:3].astype(bool), o.frozen)
        ac, av, gm = st["members"]
        assert np.array_equal(ac["H"], o.members[0].H)
        assert (av["n"], av["N_min"]) == (o.members[1].n, o.members[1].N_min)
        assert np.array_equal(av["keys"], o.members[1].keys)
        np.testing.assert_allclose(gm["mu"], o.members[2].mu, rtol=1e-9, atol=1e-9)
    assert abs(st["W"][:3].sum() - 1.0) < 1e-12


def test_single_member_portfolio_is_the_member(env):
    """Pin P11 on the GPU side: a one-member portfolio reproduces the member bit for bit."""
    torch, ile, _ = env
    N, d = 20000, 3
    a = _make(ile, "AC", d, N)
    p = _make(ile, "PORTFOLIO", d, N, members=("AC",))
    lo, hi = LO6[:d], HI6[:d]
    for it in range(3):
        za, la = a.draw(N, it)
        zp, lpp = p.draw(N, it)
        assert torch.equal(za, zp) and torch.equal(la, lpp)
        lnw = _dev(torch, _gauss_lnw(za.cpu().numpy(), lo, hi) - la.cpu().numpy())
        a.update(za, lnw, la)
        p.update(zp, lnw, lpp)
    assert np.array_equal(a.get_state()["H"], p.get_state()["members"][0]["H"])


def test_state_roundtrip(env):
    torch, ile, _ = env
    N, d = 5000, 3
    g = _make(ile, "PORTFOLIO", d, N, members=("AC", "AV", "GMM"), n_gmm=3, N_min_star=64)
    z, lp = g.draw(N, 0)
    lnw = _dev(torch, _gauss_lnw(z.cpu().numpy(), LO6[:d], HI6[:d]) - lp.cpu().numpy())
    g.update(z, lnw, lp)
    st = g.get_state()
    z1, lp1 = g.draw(N, 1)
    g.reset()
    assert g.get_state()["members"][1]["n"] == 1
    g.set_state(st)
    z2, lp2 = g.draw(N, 1)
    assert torch.equal(z1, z2) and torch.equal(lp1, lp2)


@pytest.mark.parametrize("cfg,N,n_iter", [(1, 1 << 16, 1), (2, 3000, 3), (3, 6000, 3), (5, 4000, 3)])
def test_step_parity_with_oracle(env, cfg, N, n_iter):
    """Free-running device iterations (ile_integrator_step); each iteration is checked against the
    oracle started from the same sampler state: draws, per-sample lnL (1e-9 relative), ln w,
    log-integral (1e-8), n_eff / n_ESS."""
    torch, _, _ = env
    from paper_2505_11655_b200 import Ile, Integrator, result_from_device
    from oracle.ile import IleProblem
    from oracle.integrators import make_integrator
    from oracle.reduce import reduce_lnw, combine
    prob = make_problem(cfg, N=N, n_iter=n_iter)
    ile = Ile(0)
    ile.load_problem(prob)
    g = Integrator.from_problem(ile, prob, max_batch=N)
    oo = {k: v for k, v in prob.opts.items() if k != "seed"}
    o = make_integrator(prob.kind, prob.lo, prob.hi, prob.opts["seed"], **oo)
    op = IleProblem(prob)
    parts = []
    for it in range(n_iter):
        st = g.get_state()
        if prob.kind == "PORTFOLIO":
            _load_portfolio_state(o, st)
        elif prob.kind == "AC":
            o.H, o.pi, o.cdf = st["H"].copy(), st["pi"].copy(), st["cdf"].copy()
        elif prob.kind == "AV":
            o.n, o.keys = st["n"], st["keys"].copy()
        res = result_from_device(g.step(0, N, it))[0]
        z, lp, lnL, lnw = [t.cpu().numpy() for t in g.last_batch(N)]
        zo, lpo = o.draw(N, it)
        if prob.kind != "PORTFOLIO":
            assert np.array_equal(z, zo), f"iteration {it}: draws differ"
        else:
            np.testing.assert_allclose(z, zo, rtol=0, atol=1e-9)
        ref_lp = o.ln_pdf(z) if prob.kind != "AV" else lpo
        fin = np.isfinite(ref_lp)
        np.testing.assert_allclose(lp[fin], ref_lp[fin], rtol=0, atol=1e-10)
        ref_L = op.lnL_z(z)
        ok = np.isfinite(ref_L)
        assert np.array_equal(ok, np.isfinite(lnL))
        assert np.all(np.abs(lnL[ok] - ref_L[ok]) <= 1e-9 * np.maximum(1.0, np.abs(ref_L[ok]))), np.abs(lnL[ok] - ref_L[ok]).max()
        ref_w = np.where(ok, ref_L + op.ln_prior(z) - ref_lp, -np.inf)
        ref = reduce_lnw(ref_w)
        parts.append(ref)
        assert abs(res["ln_integral"] - ref["ln_integral"]) <= 1e-8
        for k in ("n_eff", "n_ess"):
            assert abs(res[k] - ref[k]) <= 1e-7 * max(1.0, ref[k])
        cum = combine(parts)
        assert abs(res["cum_ln_integral"] - cum["ln_integral"]) <= 1e-8
        assert res["cum_n_samples"] == N * (it + 1) and res["n_samples"] == N
    if prob.kind == "AV":
        assert res["n_bins"] >= 1 and res["n_cells"] >= 1 and res["N_min"] >= 1
    if prob.kind == "PORTFOLIO":
        assert abs(res["W"][:3].sum() - 1.0) < 1e-12


def _assert_same_state(a, b, where):
    if isinstance(a, dict):
        assert a.keys() == b.keys(), where
        for k in a:
            _assert_same_state(a[k], b[k], where + (k,))
    elif isinstance(a, (list, tuple)):
        assert len(a) == len(b), where
        for q, (x, y) in enumerate(zip(a, b)):
            _assert_same_state(x, y, where + (q,))
    elif isinstance(a, np.ndarray):
        assert np.array_equal(a.view(np.uint8), b.view(np.uint8)), where
    else:
        assert a == b or (a != a and b != b), where


@pytest.mark.parametrize("cfg,N,n_iter", [(2, 40000, 4), (3, 50000, 5), (5, 30000, 5)])
def test_run_repeatable(env, cfg, N, n_iter):
    """ile_integrator_run from the reset state, again and again: every ile_result field and the final sampler state bit for
    bit the same.  The update kernels take their decisions in integers (histograms, threshold select, cell keys) and fix the
    order of every floating-point sum, so a difference is a race (e.g. in the select pass whose last block fixes the digit)."""
    torch, _, _ = env
    from paper_2505_11655_b200 import Ile, Integrator
    prob = make_problem(cfg, N=N, n_iter=n_iter)
    ile = Ile(0)
    ile.load_problem(prob)
    g = Integrator.from_problem(ile, prob, max_batch=N)
    first, first_state = None, None
    for rep in range(4):
        g.reset()
        res = g.run(0, 1, n_iter, N)
        torch.cuda.synchronize()
        raw = res.cpu().numpy().copy().view(np.uint8)
        st = g.get_state()
        if first is None:
            first, first_state = raw, st
            continue
        assert np.array_equal(first, raw), (cfg, rep)
        _assert_same_state(st, first_state, (cfg, rep))


def test_run_matches_steps_and_resets_between_points(env):
    torch, _, _ = env
    from paper_2505_11655_b200 import Ile, Integrator, result_from_device
    prob = make_problem(4, P=3, N=2048)
    ile = Ile(0)
    ile.load_problem(prob)
    g = Integrator.from_problem(ile, prob, max_batch=2048, kind="AC")
    out = result_from_device(g.run(0, 3, 2, 2048))
    assert out.shape == (6,)
    g2 = Integrator.from_problem(ile, prob, max_batch=2048, kind="AC")
    for p in range(3):
        g2.reset()
        for it in range(2):
            r = result_from_device(g2.step(p, 2048, it))[0]
            assert r["ln_integral"] == out[p * 2 + it]["ln_integral"]
            assert r["cum_ln_integral"] == out[p * 2 + it]["cum_ln_integral"]
    assert len({float(out[p * 2]["ln_integral"]) for p in range(3)}) == 3     # different intrinsic points


# ------------------------------------------------------------------------------- portfolio options of PAPER.md:297
def test_portfolio_activation_iteration_teacher_forced(env):
    """member_first_iter: two AC members with 10 and 30 bins, the second activated at iteration 3 (the paper's Fig. 7
    portfolio in small).  Same draws (bit-exact), the oracle's ln w into both updates: identical allocations,
    histograms and weights at every iteration, before, at and after the activation."""
    torch, ile, _ = env
    N, d, g0 = 40000, 4, 3
    kw = dict(members=("AC", "AC"), member_opts=[dict(n_bins=10), dict(n_bins=30)], first_iter=[0, g0])
    g = _make(ile, "PORTFOLIO", d, N, **kw)
    o = _oracle("PORTFOLIO", d, members=["AC", "AC"], member_opts=kw["member_opts"], first_iter=kw["first_iter"])
    lo, hi = LO6[:d], HI6[:d]
    for it in range(6):
        z, lp = g.draw(N, it)
        zo, lpo = o.draw(N, it)
        st = g.get_state()
        assert np.array_equal(st["alloc"][:2], o.alloc) and np.array_equal(st["active"][:2].astype(bool), o.active)
        if it < g0:
            assert st["alloc"][1] == 0 and st["W"][1] == 0.0
        zg = z.cpu().numpy()
        assert np.array_equal(zg, zo)                                        # AC draws: bit-exact
        np.testing.assert_allclose(lp.cpu().numpy(), lpo, rtol=0, atol=1e-10)
        lnw = _gauss_lnw(zg, lo, hi, width=0.08) - lpo
        o.update(zo, lnw, lpo)
        g.update(z, _dev(torch, lnw), _dev(torch, lpo))
        st = g.get_state()
        np.testing.assert_allclose(st["W"][:2], o.W, rtol=1e-11)
        assert np.array_equal(st["frozen"][:2].astype(bool)[o.active], o.frozen[o.active])
        for a in range(2):
            assert st["members"][a]["n_bins"] == (10, 30)[a]
            assert np.array_equal(st["members"][a]["H"], o.members[a].H), (it, a)
    assert st["W"][1] > 0.0


def test_portfolio_silent_member_and_estimate(env):
    """member_silent: [AC, UNIFORM (silent)]: the silent member draws N / 2 samples of every batch, the density is the
    AC member's alone, the estimate counts the contributing samples only and the AC histogram is trained on all N."""
    from paper_2505_11655_b200 import Integrand, result_from_device
    torch, ile, _ = env
    N, d = 30000, 3
    g = _make(ile, "PORTFOLIO", d, N, members=("AC", "UNIFORM"), silent=[False, True], n_bins=20)
    o = _oracle("PORTFOLIO", d, members=["AC", "UNIFORM"], silent=[False, True], n_bins=20)
    lo, hi = LO6[:d], HI6[:d]
    for it in range(3):
        z, lp = g.draw(N, it)
        zo, lpo = o.draw(N, it)
        st = g.get_state()
        assert st["alloc"][:2].tolist() == [N // 2, N // 2] == o.alloc.tolist()
        zg = z.cpu().numpy()
        assert np.array_equal(zg, zo)
        np.testing.assert_allclose(lp.cpu().numpy(), lpo, rtol=0, atol=1e-10)
        lnw = _gauss_lnw(zg, lo, hi, width=0.1) - lpo
        o.update(zo, lnw, lpo)
        g.update(z, _dev(torch, lnw), _dev(torch, lpo))
        st = g.get_state()
        assert np.array_equal(st["members"][0]["H"], o.members[0].H)          # trained on the silent samples too
        assert st["W"][:2].tolist() == [1.0, 0.0]
    # free-running step on a built-in integrand: n_samples = contributing samples; the estimate matches the closed form
    f = Integrand.gaussian_mix([[3.0, 0.0, 1.5]], [0.3], [0.0])
    g2 = _make(ile, "PORTFOLIO", d, N, members=("AC", "UNIFORM"), silent=[False, True], n_bins=40)
    for it in range(8):
        r = result_from_device(g2.step_integrand(f, N, it))[0]
    assert r["n_samples"] == N - N // 2 and r["cum_n_samples"] == 8 * (N - N // 2)
    exact = (0.3 * math.sqrt(2 * math.pi)) ** 3                              # the Gaussian sits well inside the box
    assert abs(math.exp(float(r["cum_ln_integral"])) / exact - 1) < 5 * math.sqrt(float(r["cum_rel_variance"])) + 5e-3


def test_integrator_option_validation(env):
    from paper_2505_11655_b200 import IleError
    torch, ile, _ = env
    with pytest.raises(IleError):
        _make(ile, "PORTFOLIO", 3, 1000, members=("AC", "AC"), first_iter=[1, 0])        # member 0 is always active
    with pytest.raises(IleError):
        _make(ile, "PORTFOLIO", 3, 1000, members=("AC", "UNIFORM", "AC"), silent=[False, True, False])   # silent members last
    with pytest.raises(IleError):
        _make(ile, "AC", 6, 1000, n_bins=2000)                                            # d * n_bins beyond the histogram kernel's shared memory
    with pytest.raises(IleError):
        _make(ile, "UNIFORM", 3, (1 << 24) + 1)                                           # fixed-point sums could overflow
