"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA-side tests / bench.

This module holds NONE of the method's arithmetic (no sampling, kinematics, matrix elements or
estimator): it only describes problems (species, grids, processes) and fills ``f`` arrays.  It
imports neither ``oracle`` nor ``paper_2308_04869_b200``.
"""
from .configs import KIND_CONST, KIND_COULOMB_SCREENED, KIND_TCHAN_S2, KIND_ISO_DSIGMA, make, f_layout, equilibrium_nbar  # noqa: F401
