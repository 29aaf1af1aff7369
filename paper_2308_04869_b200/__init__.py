"""B200-native Monte Carlo collision term of the RBG-Maxwell method (arXiv 2308.04869, Eq. 16-19).

Thin binding over the C ABI of ``include/rbg.h`` (``librbg.so``, built by ``paper_2308_04869_b200.build``):
argument marshalling only -- every step of the path runs in the CUDA kernels.  PyTorch supplies
device memory and streams.  There is no CPU fallback: if the library is missing or there is no
CUDA device the calls raise.
"""
from __future__ import annotations

from .binding import (  # noqa: F401
    Collision, RbgError, KIND_CONST, KIND_COULOMB_SCREENED, KIND_TCHAN_S2, KIND_ISO_DSIGMA, KIND_QCD_Q1Q2, KIND_QCD_Q1Q1, KIND_QCD_Q1QB1,
    KIND_QCD_Q1QB1_Q2QB2, KIND_QCD_QQB_GG, KIND_QCD_QG, KIND_QCD_GG, load_library, probe_alu_peak,
    exported_symbols, selftest_math, selfcheck_failures, use_checked_build, moments_static, MOMENTS_STATIC_MAX_CELLS,
)
