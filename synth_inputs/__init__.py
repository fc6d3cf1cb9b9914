"""Seeded synthetic inputs (integrals, subspace S, amplitudes psi) shared by the oracle and the CUDA path.

This module holds NONE of the method's arithmetic (no Slater-Condon rule, no screening, no phases):
it only draws random integrals / determinants / amplitudes with the recipe of BASELINE.json `configs`
and SURVEY.md section 8(d), which stand in for the paper's H2O / N2 (cc-pVDZ) and Cr2
 FCIDUMP workloads that are not available offline.
"""
from .generate import CONFIGS, make_integrals, make_subspace, make_problem, pack_index, BASE_SEED  # noqa: F401
