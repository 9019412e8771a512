"""Seeded synthetic inputs (melts) shared by the oracle-side tests and the CUDA-side tests.

This package holds NO arithmetic of the method (no forces, no neighbor search, no
integration, no random-number generator of the method): only the recipes that place beads,
bonds and velocities for the five BASELINE.json configs and the paper's two Fig. 4 liquids, plus small random
boxes for tests.
"""
from .melts import (  # noqa: F401
    CONFIGS,
    Workload,
    make_config,
    make_kg_melt,
    make_dpd_diblock,
    make_lj_liquid,
    make_dpd_liquid,
    make_random_box,
    maxwell_velocities,
)
