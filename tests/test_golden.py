"""Oracle against the golden fixtures (tests/golden/): values the paper states and what follows from them by hand."""
import json
import math
import os

import numpy as np

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _load(name):
    with open(os.path.join(GOLD, name)) as f:
        return json.load(f)


def test_fig6_mixture_integral_and_marginals():
    """the Fig. 6 mixture; its total integral and 'exact one-dimensional marginal PDFs'."""
    from oracle.integrands import gaussian_mix_box_integral, ln_gaussian_mix
    g = _load("fig6_mixture.json")
    centers, sig = g["centers"], [g["sigma"]] * 2
    box = gaussian_mix_box_integral([-60.0] * 3, [60.0] * 3, centers, sig, [0.0, 0.0])
    assert abs(box - g["integral_R3"]) <= 1e-12 * g["integral_R3"]
    # marginals of the oracle's density by 2-D trapezoid quadrature (spectrally accurate for Gaussians at h = 0.1)
    t = np.arange(-14.0, 14.0 + 1e-9, 0.1)
    A, B = np.meshgrid(t, t, indexing="ij")
    for x, p in g["x_marginal"]:
        z = np.stack([np.full(A.size, x), A.ravel(), B.ravel()])
        m = np.exp(ln_gaussian_mix(z, centers, sig, [0.0, 0.0])).sum() * 0.01 / g["integral_R3"]
        assert abs(m - p) <= 1e-10 * max(p, 1e-12), (x, m, p)
    for y, p in g["y_marginal"]:
        z = np.stack([A.ravel(), np.full(A.size, y), B.ravel()])
        m = np.exp(ln_gaussian_mix(z, centers, sig, [0.0, 0.0])).sum() * 0.01 / g["integral_R3"]
        assert abs(m - p) <= 1e-10 * p, (y, m, p)


def test_eq13_cell_refinement_cases():
    """V_{g+1}, Delta V and n_bins of Eq. 13 on hand-worked cases."""
    from oracle.integrators import AV
    g = _load("eq13_cells.json")
    for c in g["cases"]:
        d, N, N_min = c["d"], c["N_live"], c["N_min"]
        av = AV([0.0] * d, [1.0] * d, seed=1, P_thr=0.999, N_min_star=N_min)
        # a state whose live volume fraction is V_g: C cells of n^d
        if c["V_g"] == 1.0:
            pass
        elif c["V_g"] == 0.25:
            av.n, av.keys = 2, np.array([0, 1], dtype=np.uint64)          # 2 of 2^3 cells
        elif c["V_g"] == 0.001:
            av.n, av.keys = 100, np.arange(10, dtype=np.uint64)           # 10 of 100^2 cells
        assert abs(av.v - c["V_g"]) < 1e-15
        rng = np.random.Generator(np.random.Philox(7))
        z = rng.random((d, N)) * 0.999
        lnw = np.full(N, -100.0)                                          # weight 0 in fixed point ...
        lnw[:N_min] = 0.0                                                 # ... except the N_min that carry the mass
        av.update(z, lnw)
        assert av.N_min == N_min
        assert av.n == c["n_bins"], (c, av.n)


def test_portfolio_weight_floor_and_mixture_density():
    """weights follow the per-member n_ESS and never drop below 0.05 / N_s; the mixture."""
    from oracle.integrators import Portfolio
    g = _load("portfolio_floor.json")

    class Stub:
        def __init__(self, p):
            self.lo, self.hi, self.d, self.p = np.zeros(1), np.ones(1), 1, p

        def ln_pdf(self, z):
            return np.full(z.shape[1], math.log(self.p))

        def update(self, z, lnw, ln_ps):
            pass

    for c in g["cases"]:
        ness = c["n_ess"]
        P = Portfolio([Stub(1.0) for _ in ness])
        P.alloc = np.array([max(int(n), 1) for n in ness])
        lnw = np.concatenate([np.zeros(int(n)) if n >= 1 else np.full(1, -np.inf) for n in ness])   # m equal weights: n_ESS = m
        P.update(np.zeros((1, len(lnw))), lnw, np.zeros(len(lnw)))
        assert np.allclose(P.W, c["W"], rtol=1e-14, atol=0), (P.W, c["W"])
        # the floor holds for the weights before they are rescaled to sum 1 (p_s divides by sum W anyway)
        raw = np.array(ness) / np.sum(ness)
        S = np.maximum(raw, g["floor_numerator"] / len(ness)).sum()
        assert (P.W * S).min() >= g["floor_numerator"] / len(ness) * (1.0 - 1e-12)
    m = g["mixture_case"]
    P = Portfolio([Stub(p) for p in m["p"]])
    P.W = np.array(m["W"])
    assert abs(math.exp(P.ln_pdf(np.zeros((1, 1)))[0]) - m["p_s"]) < 1e-14


def test_eq7_quadratic_term_worked_case():
    """Eq. 7 with Eq. 17-18: the U/V quadratic term of a two-mode, one-detector case worked by hand."""
    from oracle.likelihood import quadratic_term
    g = _load("eq17_18_symmetry.json")
    cx = lambda a: np.array(a)[..., 0] + 1j * np.array(a)[..., 1]
    U, V, y, F = cx(g["U"])[None], cx(g["V"])[None], cx(g["y"])[:, None], np.array([[complex(*g["F"])]])
    assert np.allclose(U[0], U[0].conj().T) and np.allclose(V[0], V[0].T)          # Eq. 17-18
    B = quadratic_term(F, y, U, V)
    assert abs(B[0] - g["B"]) < 1e-15
