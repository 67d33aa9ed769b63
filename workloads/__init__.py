"""Seeded synthetic inputs (initial conditions) and the BASELINE.json configuration table.

This package serves BOTH the CUDA path and the oracle.  It holds none of the method's
arithmetic (no keys, tree, K(r), forces or integrator) -- only samplers for the particle
distributions BASELINE.json names and the parameter sets that go with them.
"""
from .ic import plummer, hernquist, cold_sphere, two_plummer, make_ic  # noqa: F401
from .configs import CONFIGS, Config, get_config, paper_params  # noqa: F401
