"""Seeded synthetic inputs + extrapolator-table design shared by the oracle tests and the CUDA path.

Holds none of the method's arithmetic: only array generators.
"""
from .configs import (make_config, sweep_point, tiny_random_problem, random_problem, random_problem_3d,  # noqa: F401
                      SWEEP_NX, SWEEP_NW, SWEEP_TAPS, BASE_SEED, NTAB)
from . import filters  # noqa: F401
