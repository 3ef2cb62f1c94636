"""Seeded synthetic inputs for the five BASELINE.json configs.

This module is shared by the CPU oracle's tests and by the CUDA path's tests and
bench.  It holds NONE of the method's arithmetic (no rates, no integrator): only
the network *descriptions* (topology + random coefficients) and the zone state
arrays (rho, T, X), built from ``numpy.random.default_rng(seed).random`` draws in
the fixed order of SURVEY.md section 8(d) / DESIGN.md "Input recipe".
"""
from .configs import (  # noqa: F401
    Network,
    Workload,
    CONFIG_NZ,
    network_for_config,
    make_workload,
    first_order_decay_network,
    aprox13_like_network,
    make_aprox13_like_workload,
    urca9_like_network,
    make_urca9_like_workload,
    sha256_of,
)
