"""Seeded synthetic DIA workloads (input data only).

This package holds the input generators shared by the CPU oracle tests, the GPU
parity tests and bench.py.  It contains none of the method's arithmetic (no
loss, noise-model-in-the-fit, gradient or optimiser code) and imports neither
`oracle/` nor the CUDA package; the simulated target image is produced with a
library correlation routine, following the paper's simulation recipe
(Section 3.1) in the shapes BASELINE.json's configs state.
"""
from .starfield import (  # noqa: F401
    CONFIGS,
    Workload,
    make_reference,
    make_target,
    make_workload,
    theta_init,
    gaussian_kernel_init,
    correlate_valid,
    n_valid,
)
