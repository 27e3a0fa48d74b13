"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This package holds NO arithmetic of the TACAW method (no potentials, no FFTs, no
propagation): only lattice builders, seeded displacement recipes, the labelled
surrogate form-factor coefficient table and the workload descriptions of
BASELINE.json `configs`.  Both `oracle/` and the CUDA path consume what it makes;
neither imports the other.
"""
from .configs import CONFIG_NAMES, Workload, make_workload  # noqa: F401
from .form_factors import form_factor_coefficients  # noqa: F401
