"""Pins of the test integrands (Fig. 6; PAPER.md:179 Rosenbrock)."""
import math

import numpy as np

from oracle.integrands import gaussian_mix_box_integral, ln_gaussian_mix, ln_rosenbrock
from oracle.integrators import make_integrator
from oracle.reduce import reduce_lnw, combine

FIG6 = dict(centers=[[4.0, 0.0, 0.0], [-4.0, 0.0, 0.0]], sigmas=[math.sqrt(2.0)] * 2, ln_amps=[0.0, 0.0])


def test_gaussian_mix_values_and_quadrature():
    z = np.array([[4.0, -4.0, 0.0], [0.0, 0.0, 0.0], [0.0, 0.0, 0.0]])
    v = ln_gaussian_mix(z, **FIG6)
    e = math.exp(-64.0 / 4.0)                                    # the other component, 8 away, sigma^2 = 2
    assert abs(v[0] - math.log(1.0 + e)) < 1e-15 and abs(v[1] - v[0]) < 1e-15
    assert abs(v[2] - math.log(2.0 * math.exp(-16.0 / 4.0))) < 1e-14
    # 1-D quadrature against the closed form (Gauss-Legendre, 400 nodes)
    x, w = np.polynomial.legendre.leggauss(400)
    lo, hi = [-10.0], [10.0]
    xs = 0.5 * (hi[0] - lo[0]) * x + 0.5 * (hi[0] + lo[0])
    one = dict(centers=[[4.0], [-4.0]], sigmas=FIG6["sigmas"], ln_amps=[0.0, math.log(0.5)])
    quad = (0.5 * (hi[0] - lo[0]) * w * np.exp(ln_gaussian_mix(xs[None, :], **one))).sum()
    assert abs(quad - gaussian_mix_box_integral(lo, hi, **one)) < 1e-12 * quad
    assert abs(gaussian_mix_box_integral([-50.0] * 3, [50.0] * 3, **FIG6) - 2.0 * (2.0 * math.pi * 2.0) ** 1.5) < 1e-9


def test_rosenbrock_values():
    z = np.array([[1.0, 0.0, -1.0], [1.0, 0.0, 2.0]])
    assert np.allclose(ln_rosenbrock(z), [0.0, -1.0, -(4.0 + 100.0)], atol=1e-15)
    assert np.allclose(ln_rosenbrock(z, T=4.0), [0.0, -0.25, -26.0], atol=1e-15)


def test_av_integrates_the_fig6_mixture():
    """Free-running oracle AV on Fig. 6's integrand: the cumulative estimate brackets the closed form."""
    lo, hi = [-10.0] * 3, [10.0] * 3
    exact = gaussian_mix_box_integral(lo, hi, **FIG6)
    av = make_integrator("AV", np.array(lo), np.array(hi), 17, N_min_star=512)
    parts = []
    for g in range(6):
        z, lp = av.draw(20000, g)
        lnw = ln_gaussian_mix(z, **FIG6) - lp
        parts.append(reduce_lnw(lnw))
        av.update(z, lnw, None)
    # after adaptation the volume misses at most 1 - P_thr of the mass: compare the last iterations
    late = combine(parts[3:])
    est = math.exp(late["ln_integral"])
    sig = est * math.sqrt(max(late["rel_variance"], 0.0))
    assert 0.99 * exact - 5 * sig <= est <= exact + 5 * sig
