"""Writes synth/injections.json: the injected-signal coefficients of each BASELINE.json config.

Calls only oracle/ (antenna patterns, harmonics) and the seeded input generators in synth/.
Run from the repo root:  python -m oracle.make_injections

For config c, theta_0 is drawn from the prior with numpy Philox(seed(c) + 500) (config 3:
inclination near edge-on, pi/2 - 0.1, "edge-on"; config 5: two templates).
Stored per template: theta_0, F_k(theta_0) = F+ - i Fx, Y_lm(iota_0, -phi_ref,0), tau_k(theta_0),
all as hex floats so the fixture is bit-reproducible.
"""
from __future__ import annotations

import json
import math
import os

import numpy as np

from oracle import likelihood as lk
from synth import workloads as wl


def main():
    out = {}
    for cfg, c in wl.CONFIGS.items():
        rng0 = np.random.Generator(np.random.Philox(wl.config_seed(cfg, 0)))
        D, pos = wl.make_network(c["K"], rng0)
        ell, m = wl.make_modes(c["lmax"])
        rng = np.random.Generator(np.random.Philox(wl.config_seed(cfg, 0) + 500))
        templates = []
        for it in range(2 if c["two_templates"] else 1):
            ra = float(rng.uniform(0.0, 2.0 * math.pi))
            dec = float(math.asin(rng.uniform(-1.0, 1.0)))
            psi = float(rng.uniform(0.0, math.pi))
            phi = float(rng.uniform(0.0, 2.0 * math.pi))
            incl = float(math.acos(rng.uniform(-1.0, 1.0)))
            if cfg == 3:
                incl = math.pi / 2.0 - 0.1
            if it == 1:                       # second template: same sky, different orientation
                ra, dec = templates[0]["theta0"]["ra"], templates[0]["theta0"]["dec"]
            Fp, Fx, tau = lk.antenna(D, pos, 0.0, np.array([ra]), np.array([dec]), np.array([psi]))
            F = (Fp - 1j * Fx)[:, 0]
            Y = lk.ylm(ell, m, np.array([incl]), np.array([-phi]))[:, 0]
            templates.append(dict(
                theta0=dict(ra=ra, dec=dec, psi=psi, phi_ref=phi, incl=incl, dist=wl.D0_MPC),
                F=[[float(v.real).hex(), float(v.imag).hex()] for v in F],
                Y=[[float(v.real).hex(), float(v.imag).hex()] for v in Y],
                tau=[float(t).hex() for t in tau[:, 0]],
            ))
        out[str(cfg)] = dict(templates=templates)
    path = os.path.join(os.path.dirname(os.path.abspath(wl.__file__)), "injections.json")
    with open(path, "w") as fh:
        json.dump(out, fh, indent=1)
    print("wrote", path)


if __name__ == "__main__":
    main()
