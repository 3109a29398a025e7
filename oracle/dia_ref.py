"""ctypes binding of oracle/libdia_ref.so (argument marshalling only)."""
from __future__ import annotations

import ctypes as C
import dataclasses
from typing import Optional

import numpy as np

from . import build as _build

LOSS_GAUSSIAN, LOSS_HUBER = 0, 1
NOISE_MODEL, NOISE_FIXED = 0, 1
FIT_STATUS = {0: "converged_grad", 1: "converged_change", 2: "max_iters", 3: "nonfinite"}


class _Config(C.Structure):
    _fields_ = [("n_rows", C.c_int), ("n_cols", C.c_int), ("m", C.c_int),
                ("loss", C.c_int), ("huber_c", C.c_double),
                ("noise", C.c_int), ("sigma0", C.c_double), ("gain", C.c_double),
                ("flat", C.c_void_p), ("lambda_reg", C.c_double), ("bg_degree", C.c_int)]


class RefFitOpts(C.Structure):
    _fields_ = [("lr_kernel", C.c_double), ("lr_b0", C.c_double),
                ("adam_beta1", C.c_double), ("adam_beta2", C.c_double), ("adam_eps", C.c_double),
                ("tol_switch", C.c_double), ("lbfgs_lr", C.c_double),
                ("lbfgs_history", C.c_int), ("lbfgs_backtrack", C.c_int),
                ("tol_change_rel", C.c_double), ("tol_grad_abs", C.c_double), ("tol_grad_rel", C.c_double),
                ("max_adam_iters", C.c_int), ("max_lbfgs_iters", C.c_int),
                ("force_adam_iters", C.c_int), ("force_lbfgs_iters", C.c_int)]

    @staticmethod
    def default(**kw) -> "RefFitOpts":
        o = RefFitOpts()
        _lib().dia_ref_default_fit_opts(C.byref(o))
        for k, v in kw.items():
            if not hasattr(o, k):
                raise AttributeError(k)
            setattr(o, k, v)
        return o


class RefFitResult(C.Structure):
    _fields_ = [("loss", C.c_double), ("grad_inf_norm", C.c_double), ("photometric_scale", C.c_double),
                ("n_adam", C.c_int), ("n_lbfgs", C.c_int), ("n_evals", C.c_int), ("status", C.c_int)]


_LIB = None


def _lib():
    global _LIB
    if _LIB is None:
        lib = C.CDLL(_build.build())
        lib.dia_ref_huber_Q.restype = C.c_double
        lib.dia_ref_huber_Q.argtypes = [C.c_double, C.c_double]
        _LIB = lib
    return _LIB


@dataclasses.dataclass
class RefConfig:
    n_rows: int
    n_cols: int
    m: int
    loss: int = LOSS_GAUSSIAN
    huber_c: float = 1.345
    noise: int = NOISE_MODEL
    sigma0: float = 5.0
    gain: float = 1.0
    flat: Optional[np.ndarray] = None
    lambda_reg: float = 0.0
    bg_degree: int = 0

    @property
    def n_params(self) -> int:
        d = self.bg_degree
        return self.m * self.m + (d + 1) * (d + 2) // 2

    def _c(self):
        keep = None
        ptr = None
        if self.flat is not None:
            keep = np.ascontiguousarray(self.flat, dtype=np.float32)
            assert keep.shape == (self.n_rows, self.n_cols)
            ptr = keep.ctypes.data
        c = _Config(self.n_rows, self.n_cols, self.m, self.loss, self.huber_c,
                    self.noise, self.sigma0, self.gain, ptr, self.lambda_reg, self.bg_degree)
        return c, keep


def _f32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float32)


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _check(rc: int, what: str):
    if rc != 0:
        raise RuntimeError(f"{what} failed with code {rc}")


def _epochs(cfg: RefConfig, I, mask, var, theta):
    I = _f32(I)
    if I.ndim == 2:
        I = I[None]
    E = I.shape[0]
    assert I.shape[1:] == (cfg.n_rows, cfg.n_cols)
    theta = _f32(theta).reshape(E, cfg.n_params)
    mask = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8).reshape(I.shape)
    var = None if var is None else _f32(var).reshape(I.shape)
    return E, I, mask, var, theta


def model(cfg: RefConfig, R, theta) -> np.ndarray:
    c, keep = cfg._c()
    R = _f32(R)
    theta = _f32(theta).reshape(-1)
    M = np.empty((cfg.n_rows - cfg.m + 1, cfg.n_cols - cfg.m + 1), dtype=np.float64)
    _check(_lib().dia_ref_model(C.byref(c), _ptr(R), _ptr(theta), _ptr(M)), "dia_ref_model")
    return M


def eval_loss_grad(cfg: RefConfig, R, I, theta, mask=None, var=None, want_scale=False):
    """-> (loss [E], grad [E][m*m+1]) and, if want_scale, S [E][m*m+1]."""
    c, keep = cfg._c()
    R = _f32(R)
    E, I, mask, var, theta = _epochs(cfg, I, mask, var, theta)
    npar = cfg.n_params
    loss = np.empty(E, dtype=np.float64)
    grad = np.empty((E, npar), dtype=np.float64)
    scale = np.empty((E, npar), dtype=np.float64) if want_scale else None
    _check(_lib().dia_ref_eval_loss_grad(C.byref(c), _ptr(R), E, _ptr(I), _ptr(mask), _ptr(var),
                                         _ptr(theta), _ptr(loss), _ptr(grad), _ptr(scale)),
           "dia_ref_eval_loss_grad")
    return (loss, grad, scale) if want_scale else (loss, grad)


def fit(cfg: RefConfig, R, I, theta0, opts: Optional[RefFitOpts] = None, mask=None, var=None):
    """-> (theta_hat float32 [E][m*m+1], list of RefFitResult)."""
    c, keep = cfg._c()
    R = _f32(R)
    E, I, mask, var, theta = _epochs(cfg, I, mask, var, theta0)
    theta = theta.copy()
    opts = opts or RefFitOpts.default()
    res = (RefFitResult * E)()
    _check(_lib().dia_ref_fit(C.byref(c), _ptr(R), C.byref(opts), E, _ptr(I), _ptr(mask), _ptr(var),
                              _ptr(theta), res), "dia_ref_fit")
    return theta, list(res)


def fit_trace(cfg: RefConfig, R, I, theta0, opts: Optional[RefFitOpts] = None, mask=None, var=None, cap=4096):
    """One epoch.  -> (theta_hat float32 [np], RefFitResult, trace_theta float64 [n_updates][np], trace_loss [n_updates]):
    the FP64 iterate after every Adam / L-BFGS update, in order."""
    c, keep = cfg._c()
    R = _f32(R)
    E, I, mask, var, theta = _epochs(cfg, I, mask, var, theta0)
    assert E == 1
    theta = theta.copy()
    opts = opts or RefFitOpts.default()
    res = RefFitResult()
    tr = np.zeros((cap, cfg.n_params), dtype=np.float64)
    trL = np.zeros(cap, dtype=np.float64)
    n = C.c_int(0)
    _check(_lib().dia_ref_fit_trace(C.byref(c), _ptr(R), C.byref(opts), _ptr(I), _ptr(mask), _ptr(var),
                                    _ptr(theta), C.byref(res), _ptr(tr), _ptr(trL), int(cap), C.byref(n)),
           "dia_ref_fit_trace")
    return theta[0], res, tr[:n.value].copy(), trL[:n.value].copy()


def b08_solve(cfg: RefConfig, R, I, mask=None, var_fixed=None, n_iters=3, clip_last=False,
              want_H=False):
    c, keep = cfg._c()
    R = _f32(R)
    I = _f32(I)
    assert I.shape == (cfg.n_rows, cfg.n_cols)
    mask = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    var_fixed = _f32(var_fixed)
    npar = cfg.m * cfg.m + 1
    theta = np.empty(npar, dtype=np.float64)
    H = np.empty((npar, npar), dtype=np.float64) if want_H else None
    _check(_lib().dia_ref_b08_solve(C.byref(c), _ptr(R), _ptr(I), _ptr(mask), _ptr(var_fixed),
                                    int(n_iters), int(bool(clip_last)), _ptr(theta), _ptr(H)),
           "dia_ref_b08_solve")
    return (theta, H) if want_H else theta


def difference_image(cfg: RefConfig, R, I, theta, mask=None, var=None):
    """-> (D float64 [n_rows][n_cols], metrics float64 [4] = N_used, MFB, MFV, chi^2) for one epoch."""
    c, keep = cfg._c()
    R, I = _f32(R), _f32(I)
    assert I.shape == (cfg.n_rows, cfg.n_cols)
    theta = _f32(theta).reshape(-1)
    mask = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    var = _f32(var)
    D = np.empty((cfg.n_rows, cfg.n_cols), dtype=np.float64)
    metrics = np.empty(4, dtype=np.float64)
    _check(_lib().dia_ref_difference_image(C.byref(c), _ptr(R), _ptr(I), _ptr(mask), _ptr(var), _ptr(theta),
                                           _ptr(D), _ptr(metrics)), "dia_ref_difference_image")
    return D, metrics


def hessian(cfg: RefConfig, R, I, theta, mask=None, var=None) -> np.ndarray:
    """-> H float64 [np][np], the Hessian of the objective at theta for one epoch."""
    c, keep = cfg._c()
    R, I = _f32(R), _f32(I)
    assert I.shape == (cfg.n_rows, cfg.n_cols)
    theta = _f32(theta).reshape(-1)
    mask = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    var = _f32(var)
    H = np.empty((cfg.n_params, cfg.n_params), dtype=np.float64)
    _check(_lib().dia_ref_hessian(C.byref(c), _ptr(R), _ptr(I), _ptr(mask), _ptr(var), _ptr(theta), _ptr(H)),
           "dia_ref_hessian")
    return H


def covariance(H, n_kernel: int):
    """-> (cov float64 [n][n], sigma float64 [n], info float64 [5]) from the Hessian H (Eq. 16-17 and the validity
    tests of PAPER.md:193); info = (valid, ln|det H|, sigma_P, min eigenvalue of cov, sign det H)."""
    H = np.ascontiguousarray(H, dtype=np.float64)
    n = H.shape[0]
    assert H.shape == (n, n)
    cov = np.empty((n, n), dtype=np.float64)
    sigma = np.empty(n, dtype=np.float64)
    info = np.empty(5, dtype=np.float64)
    _check(_lib().dia_ref_covariance(int(n), int(n_kernel), _ptr(H), _ptr(cov), _ptr(sigma), _ptr(info)),
           "dia_ref_covariance")
    return cov, sigma, info


def huber_Q(c: float, N: float) -> float:
    return float(_lib().dia_ref_huber_Q(float(c), float(N)))


def num_threads() -> int:
    return int(_lib().dia_ref_num_threads())
