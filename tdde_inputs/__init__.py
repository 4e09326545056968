"""Seeded input generators shared by the oracle, the tests and bench.py.

This package only *builds inputs* (band matrices, angular coupling matrices,
field tables, initial vectors).  It contains none of the arithmetic of the
hot path (no operator apply, no BiCGSTAB, no Crank-Nicolson step, no
preconditioner) and imports neither ``oracle`` nor the CUDA package.

Recipes: DESIGN.md section "Inputs"; SURVEY.md section 8(d) D2 (synthetic) and
8(c) C7 (hydrogen).
"""
from .problem import Problem, Term, band_to_dense, dense_to_band  # noqa: F401
from .synthetic import make_synthetic, CONFIGS, make_config  # noqa: F401
from .hydrogen import make_hydrogen  # noqa: F401
from .nondipole import make_nondipole  # noqa: F401
