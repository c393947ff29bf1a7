"""Seeded synthetic inputs for the DF-JK path (shared by the oracle tests and the CUDA path).

This module holds NONE of the method's arithmetic (no density, no J, no K, no unpacking): it only
draws the packed three-index tensor ``B[P, mu>=nu]``, the orbital coefficients ``C`` and the
occupations ``occ`` of BASELINE.json's five configs.  The recipe is stated in DESIGN.md ("Input
recipe"); the inputs stand in for the paper's real DF tensors (systems A-D),
whose geometries, PySCF and mrh are not available here.
"""
from .gen import CONFIGS, DFJKInputs, make_B_packed, make_config, make_orbitals, make_random, npair_of

__all__ = ["CONFIGS", "DFJKInputs", "make_B_packed", "make_config", "make_orbitals", "make_random", "npair_of"]
