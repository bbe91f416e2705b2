"""Seeded synthetic inputs (molecules, basis sets, densities) for the five BASELINE.json configs.

This package is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA product path
(`paper_2406_14920_b200/`).  It holds none of the method's arithmetic: no normalisation, no integrals,
no screening -- only geometry / exponent / coefficient / density draws.
"""
from .configs import Problem, make_config, subset_atoms, digest, CONFIG_SEED, ncart  # noqa: F401
