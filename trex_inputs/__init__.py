"""Seeded synthetic event generators shared by the oracle tests and the CUDA path.

This package holds NONE of the method's arithmetic (no spinors, vertices, colour
algebra, bucketing): it only draws phase-space points, flavour labels, weights and
parameter vectors, following the recipe in DESIGN.md section 4.
Both `oracle/` and `paper_2510_05100_b200/` read the arrays produced here; neither
imports the other.
"""
from .configs import (  # noqa: F401
    NTHETA, TH_ALPHA_S, TH_ALPHA_EM, TH_SIN2W, TH_MZ, TH_GAMMAZ, TH_MT, TH_GAMMAT,
    TH_CTG, TH_LAMBDA, TH_VEV, default_theta, make_config, Workload, SUBPROCESSES,
    pack_key, REX_NPOS, subprocess_by_name, subprocess_by_key, shuffled_legs,
)
from .rambo import massive_rambo  # noqa: F401
