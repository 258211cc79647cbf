"""Oracle: the paper's test integrands for the integrators (TEST INFRASTRUCTURE ONLY).

PAPER.md:261 (Fig. 6): "a superposition of two multivariate gaussians with one-dimensional standard
deviations sqrt(2), centered at (+-4, 0, 0)"; PAPER.md:179, 201, 283 (Fig. 3): "the Rosenbrock
likelihood", two-dimensional.  The paper gives no formula for the latter; the textbook Rosenbrock
function is used: ln L = -sum_i [ (a - x_i)^2 + b (x_{i+1} - x_i^2)^2 ] / T.
Plain definitions; the closed form of the Gaussian box integral is the pin (tests)."""
from __future__ import annotations

import math

import numpy as np


def ln_gaussian_mix(z, centers, sigmas, ln_amps):
    """ln sum_c exp(ln_amp_c - |z - c_c|^2 / (2 sigma_c^2)) for z [d, N] (unnormalised isotropic components)."""
    z = np.asarray(z, dtype=np.float64)
    e = []
    for c, s, la in zip(centers, sigmas, ln_amps):
        r2 = np.zeros(z.shape[1])
        for i in range(z.shape[0]):
            r2 = r2 + (z[i] - c[i]) * (z[i] - c[i])
        e.append(la - 0.5 * r2 / (s * s))
    e = np.stack(e)
    mx = e.max(axis=0)
    return mx + np.log(np.exp(e - mx).sum(axis=0))


def ln_rosenbrock(z, a=1.0, b=100.0, T=1.0):
    z = np.asarray(z, dtype=np.float64)
    s = np.zeros(z.shape[1])
    for i in range(z.shape[0] - 1):
        s = s + (a - z[i]) ** 2 + b * (z[i + 1] - z[i] * z[i]) ** 2
    return -s / T


def gaussian_mix_box_integral(lo, hi, centers, sigmas, ln_amps):
    """Closed form: sum_c amp_c prod_i sigma_c sqrt(2 pi) [Phi((hi_i - c_i)/sigma_c) - Phi((lo_i - c_i)/sigma_c)]."""
    tot = 0.0
    for c, s, la in zip(centers, sigmas, ln_amps):
        v = math.exp(la)
        for i in range(len(lo)):
            v *= s * math.sqrt(2.0 * math.pi) * 0.5 * (math.erf((hi[i] - c[i]) / (s * math.sqrt(2.0))) - math.erf((lo[i] - c[i]) / (s * math.sqrt(2.0))))
        tot += v
    return tot
