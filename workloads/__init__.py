"""Seeded synthetic input generators for the five BASELINE.json workloads.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA library
(``paper_1103_4887_b200/``) with identical arrays.  It contains none of the
method's arithmetic: no action, no Delta-A, no Metropolis rule, no Philox.  The
only model code here is a numpy integrator used to SYNTHESISE the observation
series y (the "twin experiment" data of PAPER.md:272, 278), which is an input
to the method, not part of it.  Neither ``oracle/`` nor the CUDA package calls
that integrator for anything they compute.
"""
from .configs import (  # noqa: F401
    MODEL_LINEAR, MODEL_HH, MODEL_HH_CLASSIC, HH_P_TRUE, Workload, make_workload, hh_truth, linear_truth,
    linear_matrix, N_CONFIGS, lorenz_current, PAPER_P_TRUE,
)
