"""Seeded synthetic input generators shared by the oracle-side tests and the CUDA path.

Nothing in this sub-package implements a step of the method (no ray trace, sweep, harmonics of
directions, source construction or dose weighting): it only produces the tables and grids that are
arguments of `dos_create` / `dos_uncollided`.
"""
from . import configs, phantoms, quadrature, xs  # noqa: F401
from .configs import make_problem, n_updates, scan_source  # noqa: F401
