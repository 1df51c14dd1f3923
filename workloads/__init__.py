"""Seeded synthetic TDA-risp workloads (inputs only; no method arithmetic).

Shared by the oracle, the CUDA binding's tests and bench.py.  Nothing here
computes an electron-repulsion integral, a sigma vector or an eigenvalue: the
module only draws geometries, basis-set numbers, MO coefficients, orbital
energies and trial vectors with the shapes of the paper's workloads
(BASELINE.json `configs`; recipe in DESIGN.md).
"""
from .generate import make_system, trial_vectors, CONFIG_NAMES, BASE_SEED, HARTREE_EV, BOHR_ANG  # noqa: F401
