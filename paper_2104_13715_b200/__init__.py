"""B200-native DIA objective/gradient/fit engine (hot path of arxiv 2104.13715, PyTorchDIA).

Thin Python binding over the C ABI of include/dia.h (libdia_b200.so, hand-written sm_100a
kernels).  There is no CPU fallback: using the engine without the built extension or without
a CUDA device raises.
"""
from .binding import (  # noqa: F401
    DiaError,
    FitOpts,
    FitResult,
    Handle,
    dia_create,
    dia_destroy,
    dia_difference_image,
    dia_hessian,
    dia_covariance,
    dia_eval_loss_grad,
    dia_eval_loss_grad_static,
    STATIC_SCRATCH_BYTES,
    dia_fit,
    dia_fit_host,
    dia_eval_loss_grad_host,
    dia_measure_fp32_peak,
    dia_measure_fp32_pattern,
    dia_tc_probe_gemm,
    dia_hess_tc_plan,
    load_library,
    LOSS_GAUSSIAN,
    LOSS_HUBER,
    NOISE_MODEL,
    NOISE_FIXED,
    FIT_STATUS,
    EXPORTED_SYMBOLS,
)
