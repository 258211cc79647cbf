"""Writes the golden fixtures of this directory: the paper's stated values and the hand arithmetic that follows.

Plain Python arithmetic only: nothing here imports `oracle/` or the CUDA path.  Run from the repository root:
    python tests/golden/make_golden.py
"""
import json
import math
import os

HERE = os.path.dirname(os.path.abspath(__file__))


def dump(name, obj):
    with open(os.path.join(HERE, name), "w") as f:
        json.dump(obj, f, indent=1)


def fig6():
    s2 = math.sqrt(2.0)
    total = 2.0 * (2.0 * math.pi * 2.0) ** 1.5               # two unit-amplitude Gaussians, variance 2, in 3-D

    def n1(x, mu):
        return math.exp(-(x - mu) ** 2 / 4.0) / math.sqrt(4.0 * math.pi)

    dump("fig6_mixture.json", {
        "citation": "PAPER.md:261, Fig. 6 caption: 'a superposition of two multivariate gaussians with one-dimensional standard deviations sqrt(2), centered at (+-4, 0, 0)'; 'the solid blue lines on the diagonal show the exact one-dimensional marginal PDFs'",
        "sigma": s2, "centers": [[4.0, 0.0, 0.0], [-4.0, 0.0, 0.0]],
        "arithmetic": "integral over R^3 of exp(-|z-c1|^2/(2 sigma^2)) + exp(-|z-c2|^2/(2 sigma^2)) = 2 (2 pi sigma^2)^(3/2) = 2 (4 pi)^(3/2); normalised x-marginal p(x) = [N(x; 4, 2) + N(x; -4, 2)] / 2, y- and z-marginals N(0, 2)",
        "integral_R3": total,
        "x_marginal": [[x, 0.5 * (n1(x, 4.0) + n1(x, -4.0))] for x in (-6.0, -4.0, -2.0, 0.0, 1.0, 4.0, 5.5)],
        "y_marginal": [[y, n1(y, 0.0)] for y in (-3.0, 0.0, 0.5, 2.0)],
    })


def eq13():
    cases = []
    for (Vg, Nmin, Nlive, d) in [(1.0, 10000, 100000, 2), (1.0, 4096, 65536, 6), (0.25, 2500, 10000, 3), (1.0, 1, 1, 1), (0.001, 40000, 50000, 2)]:
        V1 = Vg * Nmin / Nlive
        dV = V1 / math.sqrt(Nmin)
        x = 1.0 / dV
        n = int(math.floor(x ** (1.0 / d) + 1e-9))
        while (n + 1) ** d <= x * (1 + 1e-12):
            n += 1
        while n ** d > x * (1 + 1e-12):
            n -= 1
        cases.append({"V_g": Vg, "N_min": Nmin, "N_live": Nlive, "d": d, "V_next": V1, "Delta_V": dV, "one_over_Delta_V": x, "n_bins": max(n, 1)})
    dump("eq13_cells.json", {
        "citation": "PAPER.md:265-270: V_{g+1} = V_g N_min / N_live; Delta V_{g+1} = V_{g+1} / sqrt(N_min); n_bins = (1 / Delta V_{g+1})^(1/d) (Eq. 13), taken as the largest integer whose d-th power does not exceed 1 / Delta V (reading G22)",
        "arithmetic": "e.g. V_g = 1, N_min = 10000, N_live = 100000, d = 2: V = 0.1, Delta V = 0.1 / 100 = 0.001, 1 / Delta V = 1000, n_bins = floor(sqrt(1000)) = 31",
        "cases": cases})


def portfolio():
    dump("portfolio_floor.json", {
        "citation": "PAPER.md:297: 'These weights will evolve but can never drop below 0.05/N_s where N_s is the number of members'; PAPER.md:289: p_s(x) = [sum_a W_a p_s,a(x)] / sum_a W_a",
        "floor_numerator": 0.05,
        "arithmetic": "N_s = 3, per-member n_ESS = (900, 99, 1): raw = (0.9, 0.099, 0.001); floor 0.05/3 = 0.016667 lifts the third: (0.9, 0.099, 0.016667) / 1.015667; N_s = 2, n_ESS = (1, 1): (0.5, 0.5); n_ESS = (10, 0): (1, 0.025) / 1.025",
        "cases": [
            {"n_ess": [900.0, 99.0, 1.0], "W": [0.9 / (0.999 + 0.05 / 3), 0.099 / (0.999 + 0.05 / 3), (0.05 / 3) / (0.999 + 0.05 / 3)]},
            {"n_ess": [1.0, 1.0], "W": [0.5, 0.5]},
            {"n_ess": [10.0, 0.0], "W": [1.0 / 1.025, 0.025 / 1.025]}],
        "mixture_case": {"W": [0.75, 0.25], "p": [2.0, 6.0], "p_s": 3.0}})


def eq7():
    U = [[2.0 + 0j, 0.5 - 0.25j], [0.5 + 0.25j, 1.0 + 0j]]            # Hermitian (Eq. 17)
    V = [[0.3 + 0.1j, -0.2 + 0.4j], [-0.2 + 0.4j, 0.1 - 0.3j]]          # symmetric (Eq. 18)
    y = [0.6 - 0.2j, -0.1 + 0.7j]
    F = 0.4 - 0.3j
    yUy = sum(y[a].conjugate() * U[a][b] * y[b] for a in range(2) for b in range(2))
    yVy = sum(y[a] * V[a][b] * y[b] for a in range(2) for b in range(2))
    B = 0.25 * (abs(F) ** 2 * yUy.real + (F * F * yVy).real)
    dump("eq17_18_symmetry.json", {
        "citation": "PAPER.md:78-87 (Eq. 6b-c), Eq. 7 and Eq. 17-18: B = 1/4 sum_k [ |F_k|^2 Re(y^H U_k y) + Re(F_k^2 y^T V_k y) ] with U Hermitian and V symmetric",
        "arithmetic": "one detector, two modes; y^H U y and y^T V y summed term by term in complex arithmetic",
        "U": [[[z.real, z.imag] for z in row] for row in U], "V": [[[z.real, z.imag] for z in row] for row in V],
        "y": [[z.real, z.imag] for z in y], "F": [F.real, F.imag],
        "yHUy": [yUy.real, yUy.imag], "yTVy": [yVy.real, yVy.imag], "B": B})


if __name__ == "__main__":
    fig6()
    eq13()
    portfolio()
    eq7()
