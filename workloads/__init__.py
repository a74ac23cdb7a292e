"""Seeded synthetic inputs shared by the oracle and the CUDA path.

This package holds ONLY input recipes (closed-form met fields, sources, grids,
constants of the five BASELINE.json configs).  It contains none of the method's
arithmetic (no RNG, no interpolation, no stepping, no binning) and imports
neither ``oracle`` nor ``paper_0912_3223_b200``.  Recipe: DESIGN.md §4
(from SURVEY.md §8(d)).
"""
from .configs import Workload, Nuclide, Grid, RainBox, Release, make, NAMES  # noqa: F401
