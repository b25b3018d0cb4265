"""Seeded synthetic workload generators (BASELINE.json:configs[0..4]).

This package produces *data only* (geometry, h, L, Psi, Phi).  It holds none of the
LO-AFQMC arithmetic, and is the one module both the CPU oracle's tests and the CUDA
path's tests/bench share.  See DESIGN.md "Input recipe".
"""
from .configs import (CONFIGS, CasTrial, Problem, make_cas_trial, make_problem, make_problem_from_geometry, make_walkers,  # noqa: F401
                      site_geometry, chain_geometry,
                      random_orthogonal)
