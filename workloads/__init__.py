"""Seeded synthetic inputs shared by the tests, the oracle harness and bench.py.

This package holds NO arithmetic of the method (no force law, no integrator,
no Roche formula): only the recipes that lay out two stars of elements, as
DESIGN.md "Input recipe" states them.  Both the CUDA path and the CPU oracle
consume the float32 arrays produced here.
"""
from .configs import (CONFIGS, SCENARIOS, make_config, make_binary, make_scenario, params_f32,  # noqa: F401
                      Workload)
