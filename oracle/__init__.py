"""CPU oracle for the DIA hot path -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It never imports the CUDA package.
"""
from .dia_ref import (  # noqa: F401
    RefConfig,
    RefFitOpts,
    RefFitResult,
    eval_loss_grad,
    fit,
    fit_trace,
    b08_solve,
    difference_image,
    hessian,
    covariance,
    model,
    huber_Q,
    num_threads,
    LOSS_GAUSSIAN,
    LOSS_HUBER,
    NOISE_MODEL,
    NOISE_FIXED,
)
