"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA-side harness.

This module holds NONE of the method's arithmetic: no Gaussian integrals, no A matrix, no
propagator.  It draws geometries, shell tables, orthogonal matrices, orbital energies, trial
vectors and pulse parameters from numpy's PCG64, with the recipe of BASELINE.json `configs`
under the readings R11-R18 listed in DESIGN.md.  The overlap matrix S needed for
C = S^-1/2 Q is an INPUT here (computed by whichever side is running), never computed here.
"""
from .molecules import (Basis, Config, CONFIGS, SEED, make_basis, make_mos, make_vectors,
                        get_config, orthonormalizer)

__all__ = ["Basis", "Config", "CONFIGS", "SEED", "make_basis", "make_mos", "make_vectors",
           "get_config", "orthonormalizer"]
