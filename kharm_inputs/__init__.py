"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

This package holds PROBLEM DEFINITIONS only (initial conditions, parameter sets, the
counter-based RNG).  It imports neither `oracle` nor `paper_2408_01361_b200`, and none of the
scheme's arithmetic (reconstruction, fluxes, Flux-CT, U->P, floors, ...) lives here.  The
coordinate/metric formulas it needs to *pose* the problems (Kerr-Schild, FMKS) are written in
numpy here, independently of both implementations.

The paper's EHT-library data and parameter files are not available; these inputs stand in for
them with the shapes, value ranges and structure BASELINE.json's `configs` describe.  The
recipes are stated in DESIGN.md ("Input recipe").
"""
from .params import base_params, config_params, NG, PRIM_NAMES  # noqa: F401
from .rng import splitmix64_uniform  # noqa: F401
from . import geometry, modes, bondi, torus  # noqa: F401
