"""Seeded synthetic input generators shared by the oracle, the tests and bench.py.

Holds none of the method's arithmetic (no sampling, lifting, rollout, safe test or selection);
see DESIGN.md section 4 for the recipe.
"""
from .generate import Workload, make, CONFIG_NAMES, tick_inputs  # noqa: F401
