"""Seeded synthetic workloads (inputs only) shared by the oracle tests, the GPU
parity tests and bench.py.  This package holds NO projection arithmetic: it
only manufactures the five BASELINE.json input sets (grids, initial conditions,
scheme solutions `u_true`, noisy fields `u_hat`).  Neither `oracle/` nor the CUDA
path is imported from here.
"""
from .generators import (  # noqa: F401
    KIND_HEAT1D_IC_MASS, KIND_BURGERS1D_LF, KIND_FISHER1D_IE,
    KIND_ALLENCAHN2D_IE, KIND_BURGERS1D_LF_MASS, KIND_NAMES,
    Workload, make_workload, default_params, burgers_tau_input, CONFIG_SHAPES,
)
