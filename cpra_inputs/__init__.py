"""Seeded synthetic input generators for the CPRA loop (no method arithmetic; see generate.py)."""
from .generate import (CONFIGS, Problem, angles_for, build_projector, make_object, make_problem,
                       project, project_numpy, random_phase_estimate,
                       random_stack)

__all__ = ["CONFIGS", "Problem", "angles_for", "build_projector", "make_object", "make_problem",
           "project", "project_numpy", "random_phase_estimate", "random_stack"]
