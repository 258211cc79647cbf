"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

This package builds *inputs only* (detector tensors, mode lists, U/V Gram matrices,
Q time series, time grids, prior boxes, a distance-marginalisation table).  It holds
none of the method's evaluation arithmetic (no antenna patterns, no spherical
harmonics, no likelihood, no integrator step): the injected-signal coefficients it
needs are read from ``injections.json``, a fixture written by
``oracle/make_injections.py`` (which calls only ``oracle/`` and this package).

Recipe: SURVEY.md section 8(d), restated in DESIGN.md section 4.
"""
from .workloads import (  # noqa: F401
    C_LIGHT, FS, Problem, config_seed, make_modes, make_network, make_uv, make_q,
    make_problem, make_distance_table, load_injection, CONFIGS,
)
