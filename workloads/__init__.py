"""Seeded synthetic LP inputs shared by the oracle tests, the GPU tests and bench.py.

This package holds NO arithmetic of the PDHG method (no preconditioning, no
step, no residual): it only builds problem data

    min c'x  s.t.  A x {=,>=} b,  l <= x <= u          (BASELINE.json north_star)

as host numpy arrays in the layout the C ABI takes (CSR, 0-based, int64 row
pointers, int32 column indices, fp64 values, sense bytes 'E'/'G').

Recipes: DESIGN.md "Input recipe" (restating SURVEY.md 8(d) / BASELINE.json configs[0..4]).
The paper's ARPA-E GO-Challenge-3 6,049-bus dataset (ref [16] l.279) is
not available; the UC LPs below take its shape and stand in for it.
"""
from .lp import LP
from .uc_lp import uc_lp, UC_CONFIGS, uc_config, fix_commitment
from .random_lp import random_lp, SWEEP_SIZES, sweep_config
from . import tiny

__all__ = ["LP", "uc_lp", "UC_CONFIGS", "uc_config", "fix_commitment",
           "random_lp", "SWEEP_SIZES", "sweep_config", "tiny"]
