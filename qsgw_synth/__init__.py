"""Seeded synthetic workloads for the chi0(q, i*omega) build.

This package holds ONLY input generation (shapes, random draws, occupations that
are *inputs* at the C-ABI boundary).  It contains none of the method's arithmetic
(no z, no pair weights, no chi0) and is the only module shared by the oracle
tests, the CUDA parity tests and bench.py.  Recipe: DESIGN.md section "Inputs".
"""
from .configs import CONFIGS, WorkloadConfig, get_config, scaled_config
from .ipw import IpwProblem, synthetic_ipw
from .generate import Problem, SpinChannel, coulomb_eigenvalues, binned_pair_weights, generate, haar_unitary, log_bin_edges, synthetic_mpb_matrices, synthetic_wc

__all__ = [
    "CONFIGS", "WorkloadConfig", "get_config", "scaled_config",
    "Problem", "SpinChannel", "generate", "haar_unitary", "coulomb_eigenvalues", "synthetic_wc", "binned_pair_weights", "log_bin_edges", "IpwProblem", "synthetic_ipw", "synthetic_mpb_matrices",
]
