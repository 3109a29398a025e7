"""ctypes binding of libdia_b200.so -- argument marshalling only.

The functions mirror include/dia.h one to one (dia_create, dia_eval_loss_grad, dia_fit,
dia_destroy); `Handle` is a small convenience wrapper that allocates the outputs as torch
CUDA tensors.  PyTorch is used for device memory and streams only.
"""
from __future__ import annotations

import contextlib
import ctypes as C
import os
from typing import Optional

import torch

from . import build as _build

LOSS_GAUSSIAN, LOSS_HUBER = 0, 1
NOISE_MODEL, NOISE_FIXED = 0, 1
FIT_STATUS = {0: "converged_grad", 1: "converged_change", 2: "max_iters", 3: "nonfinite"}
EXPORTED_SYMBOLS = ("dia_default_fit_opts", "dia_create", "dia_eval_loss_grad", "dia_fit",
                    "dia_destroy", "dia_status_string", "dia_last_error", "dia_get_info",
                    "dia_measure_fp32_peak", "dia_measure_fp32_pattern", "dia_difference_image", "dia_hessian", "dia_covariance",
                    "dia_eval_loss_grad_static", "dia_tc_probe_gemm", "dia_eval_loss_grad_host", "dia_fit_host", "dia_hess_tc_plan")
STATIC_SCRATCH_BYTES = 4 << 20          # DIA_STATIC_SCRATCH_BYTES of include/dia.h


class DiaError(RuntimeError):
    pass


_NO_CTX = contextlib.nullcontext()


class _Config(C.Structure):
    _fields_ = [("n_rows", C.c_int), ("n_cols", C.c_int), ("m", C.c_int), ("max_epochs", C.c_int),
                ("loss", C.c_int), ("huber_c", C.c_float),
                ("noise", C.c_int), ("sigma0", C.c_float), ("gain", C.c_float),
                ("d_flat", C.c_void_p), ("stream", C.c_void_p), ("n_refs", C.c_int), ("lambda_reg", C.c_float), ("bg_degree", C.c_int)]


class FitOpts(C.Structure):
    _fields_ = [("lr_kernel", C.c_float), ("lr_b0", C.c_float),
                ("adam_beta1", C.c_double), ("adam_beta2", C.c_double), ("adam_eps", C.c_double),
                ("tol_switch", C.c_double), ("lbfgs_lr", C.c_double),
                ("lbfgs_history", C.c_int), ("lbfgs_backtrack", C.c_int),
                ("tol_change_rel", C.c_double), ("tol_grad_abs", C.c_double), ("tol_grad_rel", C.c_double),
                ("max_adam_iters", C.c_int), ("max_lbfgs_iters", C.c_int),
                ("force_adam_iters", C.c_int), ("force_lbfgs_iters", C.c_int)]

    @staticmethod
    def default(**kw) -> "FitOpts":
        o = FitOpts()
        load_library().dia_default_fit_opts(C.byref(o))
        for k, v in kw.items():
            if not hasattr(o, k):
                raise AttributeError(k)
            setattr(o, k, v)
        return o


class FitResult(C.Structure):
    _fields_ = [("loss", C.c_double), ("grad_inf_norm", C.c_double), ("photometric_scale", C.c_double),
                ("n_adam", C.c_int), ("n_lbfgs", C.c_int), ("n_evals", C.c_int), ("status", C.c_int)]


_LIB = None


def load_library(build_if_missing: bool = True):
    """Loads libdia_b200.so (building it with nvcc if it is missing or stale).  Raises if it
    cannot be loaded: there is no fallback implementation."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = _build.LIB
    if build_if_missing and os.environ.get("DIA_NO_BUILD") != "1":
        try:
            path = _build.build()
        except Exception as exc:  # stale-but-present library is still usable
            if not os.path.exists(path):
                raise DiaError(f"cannot build {path}: {exc}") from exc
    if not os.path.exists(path):
        raise DiaError(f"{path} is missing; run python -m paper_2104_13715_b200.build")
    lib = C.CDLL(path)
    lib.dia_status_string.restype = C.c_char_p
    lib.dia_status_string.argtypes = [C.c_int]
    lib.dia_last_error.restype = C.c_char_p
    lib.dia_last_error.argtypes = [C.c_void_p]
    lib.dia_create.argtypes = [C.POINTER(_Config), C.c_void_p, C.POINTER(C.c_void_p)]
    lib.dia_eval_loss_grad.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p,
                                       C.c_void_p, C.c_void_p, C.c_void_p]
    lib.dia_eval_loss_grad_static.argtypes = [C.POINTER(_Config), C.c_void_p, C.c_int] + [C.c_void_p] * 6
    lib.dia_fit.argtypes = [C.c_void_p, C.POINTER(FitOpts), C.c_int, C.c_void_p, C.c_void_p, C.c_void_p,
                            C.c_void_p, C.c_void_p]
    lib.dia_destroy.argtypes = [C.c_void_p]
    lib.dia_difference_image.argtypes = [C.c_void_p, C.c_int] + [C.c_void_p] * 6
    lib.dia_hessian.argtypes = [C.c_void_p] * 6
    lib.dia_covariance.argtypes = [C.c_void_p] * 5
    lib.dia_get_info.argtypes = [C.c_void_p] + [C.POINTER(C.c_int)] * 4
    lib.dia_measure_fp32_peak.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
    lib.dia_measure_fp32_pattern.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_double)]
    lib.dia_eval_loss_grad_host.argtypes = [C.c_void_p, C.c_int] + [C.c_void_p] * 4
    lib.dia_fit_host.argtypes = [C.c_void_p, C.POINTER(FitOpts), C.c_int] + [C.c_void_p] * 4 + [C.c_int]
    lib.dia_hess_tc_plan.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int), C.c_void_p, C.c_int, C.c_void_p, C.c_int]
    lib.dia_tc_probe_gemm.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int]
    _LIB = lib
    return lib


def _dptr(t: Optional[torch.Tensor], dtype, what: str):
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise DiaError(f"{what} must be a contiguous CUDA tensor of dtype {dtype}")
    return C.c_void_p(t.data_ptr())


def _check(rc: int, handle=None):
    if rc != 0:
        lib = load_library()
        msg = lib.dia_last_error(handle).decode()
        raise DiaError(f"{lib.dia_status_string(rc).decode()} ({rc}): {msg}")


# ------------------------------------------------------------------------------------------
# one-to-one C ABI
# ------------------------------------------------------------------------------------------
def dia_create(n_rows: int, n_cols: int, m: int, d_R: torch.Tensor, *, max_epochs: int = 1,
               loss: int = LOSS_GAUSSIAN, huber_c: float = 1.345, noise: int = NOISE_MODEL,
               sigma0: float = 0.0, gain: float = 1.0, d_flat: Optional[torch.Tensor] = None,
               stream: Optional[torch.cuda.Stream] = None, n_refs: int = 1, lambda_reg: float = 0.0,
               bg_degree: int = 0) -> int:
    lib = load_library()
    cfg = _Config(n_rows, n_cols, m, max_epochs, loss, huber_c, noise, sigma0, gain,
                  None if d_flat is None else _dptr(d_flat, torch.float32, "d_flat").value,
                  None if stream is None else stream.cuda_stream, n_refs, lambda_reg, bg_degree)
    want = (n_rows, n_cols) if n_refs <= 1 else (n_refs, n_rows, n_cols)
    if d_R is not None and tuple(d_R.shape) != want:
        raise DiaError("d_R has the wrong shape")
    out = C.c_void_p()
    _check(lib.dia_create(C.byref(cfg), _dptr(d_R, torch.float32, "d_R"), C.byref(out)))
    return out.value


def dia_eval_loss_grad(handle: int, n_epochs: int, d_I, d_mask, d_var, d_theta, d_loss, d_grad) -> None:
    lib = load_library()
    _check(lib.dia_eval_loss_grad(handle, n_epochs, _dptr(d_I, torch.float32, "d_I"),
                                  _dptr(d_mask, torch.uint8, "d_mask"), _dptr(d_var, torch.float32, "d_var"),
                                  _dptr(d_theta, torch.float32, "d_theta"),
                                  _dptr(d_loss, torch.float64, "d_loss"), _dptr(d_grad, torch.float64, "d_grad")),
           handle)


def dia_eval_loss_grad_static(n_rows: int, n_cols: int, m: int, d_R, n_epochs: int, d_I, d_mask, d_var, d_theta,
                              d_loss, d_grad, *, loss: int = LOSS_GAUSSIAN, huber_c: float = 1.345,
                              noise: int = NOISE_MODEL, sigma0: float = 0.0, gain: float = 1.0, d_flat=None,
                              stream: Optional[torch.cuda.Stream] = None, n_refs: int = 1, lambda_reg: float = 0.0,
                              bg_degree: int = 0) -> None:
    """dia_eval_loss_grad without a handle and without any device allocation: the block partials go to the
    library's static device array (at most STATIC_SCRATCH_BYTES; include/dia.h).  All arguments are the caller's
    tensors; calls that can overlap on the GPU race on the array."""
    lib = load_library()
    cfg = _Config(n_rows, n_cols, m, n_epochs, loss, huber_c, noise, sigma0, gain,
                  None if d_flat is None else _dptr(d_flat, torch.float32, "d_flat").value,
                  None if stream is None else stream.cuda_stream, n_refs, lambda_reg, bg_degree)
    _check(lib.dia_eval_loss_grad_static(C.byref(cfg), _dptr(d_R, torch.float32, "d_R"), n_epochs,
                                         _dptr(d_I, torch.float32, "d_I"), _dptr(d_mask, torch.uint8, "d_mask"),
                                         _dptr(d_var, torch.float32, "d_var"), _dptr(d_theta, torch.float32, "d_theta"),
                                         _dptr(d_loss, torch.float64, "d_loss"), _dptr(d_grad, torch.float64, "d_grad")))


def dia_tc_probe_gemm(d_A: torch.Tensor, d_B: torch.Tensor, mode: int) -> torch.Tensor:
    """Tensor-core probe (measurement only): D [128][N] = A [128][K] @ B [N][K]' on one CTA, operands and accumulation as
    in dia_hessian's tensor-core kernel; mode 0 float16, 1 float16 hi + lo split, 2 tf32, 3 tf32 split."""
    lib = load_library()
    K, N = int(d_A.shape[1]), int(d_B.shape[0])
    if tuple(d_A.shape) != (128, K) or tuple(d_B.shape) != (N, K):
        raise DiaError("d_A must be [128][K] and d_B [N][K]")
    d_D = torch.empty((128, N), dtype=torch.float32, device=d_A.device)
    _check(lib.dia_tc_probe_gemm(None, _dptr(d_A, torch.float32, "d_A"), _dptr(d_B, torch.float32, "d_B"),
                                 _dptr(d_D, torch.float32, "d_D"), K, N, mode))
    return d_D


def _hptr(t: Optional[torch.Tensor], dtype, what: str):
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise DiaError(f"{what} must be a contiguous HOST tensor of dtype {dtype}")
    return C.c_void_p(t.data_ptr())


def dia_eval_loss_grad_host(handle: int, n_epochs: int, h_I, h_theta, h_loss, h_grad) -> None:
    lib = load_library()
    _check(lib.dia_eval_loss_grad_host(handle, n_epochs, _hptr(h_I, torch.float32, "h_I"), _hptr(h_theta, torch.float32, "h_theta"),
                                       _hptr(h_loss, torch.float64, "h_loss"), _hptr(h_grad, torch.float64, "h_grad")), handle)


def dia_fit_host(handle: int, opts: FitOpts, n_epochs: int, h_I, h_mask, h_theta, h_result, chunks: int = 0) -> None:
    lib = load_library()
    _check(lib.dia_fit_host(handle, C.byref(opts), n_epochs, _hptr(h_I, torch.float32, "h_I"), _hptr(h_mask, torch.uint8, "h_mask"),
                            _hptr(h_theta, torch.float32, "h_theta"), _hptr(h_result, torch.uint8, "h_result"), chunks), handle)


def dia_hess_tc_plan(m: int, bg_degree: int = 0):
    """Work plan of dia_hessian's tensor-core kernel (host arithmetic, no device): (n_groups, types [n][5] uint8 =
    g0, g1, a_sel, b_start, b_groups, perm [128 n_groups] int16 = parameter of every operand slot, -1 = empty)."""
    import numpy as np
    lib = load_library()
    G, n = C.c_int(), C.c_int()
    types = np.zeros((160, 5), dtype=np.uint8)
    perm = np.zeros(128 * 32, dtype=np.int16)
    _check(lib.dia_hess_tc_plan(m, bg_degree, C.byref(G), C.byref(n), types.ctypes.data_as(C.c_void_p), 160,
                                perm.ctypes.data_as(C.c_void_p), perm.size))
    return G.value, types[:n.value].copy(), perm[:128 * G.value].copy()


def dia_fit(handle: int, opts: FitOpts, n_epochs: int, d_I, d_mask, d_var, d_theta, d_result) -> None:
    lib = load_library()
    _check(lib.dia_fit(handle, C.byref(opts), n_epochs, _dptr(d_I, torch.float32, "d_I"),
                       _dptr(d_mask, torch.uint8, "d_mask"), _dptr(d_var, torch.float32, "d_var"),
                       _dptr(d_theta, torch.float32, "d_theta"), _dptr(d_result, torch.uint8, "d_result")),
           handle)


def dia_difference_image(handle: int, n_epochs: int, d_I, d_mask, d_var, d_theta, d_D, d_metrics) -> None:
    lib = load_library()
    _check(lib.dia_difference_image(handle, n_epochs, _dptr(d_I, torch.float32, "d_I"),
                                    _dptr(d_mask, torch.uint8, "d_mask"), _dptr(d_var, torch.float32, "d_var"),
                                    _dptr(d_theta, torch.float32, "d_theta"), _dptr(d_D, torch.float32, "d_D"),
                                    _dptr(d_metrics, torch.float64, "d_metrics")), handle)


def dia_hessian(handle: int, d_I, d_mask, d_var, d_theta, d_H) -> None:
    lib = load_library()
    _check(lib.dia_hessian(handle, _dptr(d_I, torch.float32, "d_I"), _dptr(d_mask, torch.uint8, "d_mask"),
                           _dptr(d_var, torch.float32, "d_var"), _dptr(d_theta, torch.float32, "d_theta"),
                           _dptr(d_H, torch.float64, "d_H")), handle)


def dia_covariance(handle: int, d_H, d_cov, d_sigma, d_info) -> None:
    lib = load_library()
    _check(lib.dia_covariance(handle, _dptr(d_H, torch.float64, "d_H"), _dptr(d_cov, torch.float64, "d_cov"),
                              _dptr(d_sigma, torch.float64, "d_sigma"), _dptr(d_info, torch.float64, "d_info")), handle)


def dia_destroy(handle: int) -> None:
    _check(load_library().dia_destroy(handle))


def dia_measure_fp32_peak(stream: Optional[torch.cuda.Stream] = None) -> float:
    """Measured FP32 peak of the current device in FMA/s (register-only FFMA microbenchmark)."""
    out = C.c_double()
    _check(load_library().dia_measure_fp32_peak(None if stream is None else stream.cuda_stream, C.byref(out)))
    return out.value


def dia_measure_fp32_pattern(pattern: int, stream: Optional[torch.cuda.Stream] = None) -> float:
    """FMA/s of one operand pattern of the register-only microbenchmark (include/dia.h): 0 pipe peak, 1 forward
    stencil (FFMA2, uniform multiplicand), 2 gradient (FFMA2, vector operands), 3 scalar three-register FFMA."""
    out = C.c_double()
    _check(load_library().dia_measure_fp32_pattern(None if stream is None else stream.cuda_stream, int(pattern), C.byref(out)))
    return out.value


# ------------------------------------------------------------------------------------------
# convenience wrapper
# ------------------------------------------------------------------------------------------
class Handle:
    """Owns one dia_handle and keeps the borrowed tensors (R, flat) alive."""

    def __init__(self, R: torch.Tensor, m: int, *, max_epochs: int = 1, loss: int = LOSS_GAUSSIAN,
                 huber_c: float = 1.345, noise: int = NOISE_MODEL, sigma0: float = 0.0, gain: float = 1.0,
                 flat: Optional[torch.Tensor] = None, stream: Optional[torch.cuda.Stream] = None,
                 lambda_reg: float = 0.0, bg_degree: int = 0):
        """R [n_rows][n_cols]: one reference shared by all epochs; R [max_epochs][n_rows][n_cols] (3-D): one
        reference per epoch (many independent image pairs fitted together)."""
        self.R, self.flat, self.m, self.max_epochs = R, flat, m, max_epochs
        self.n_refs = 1
        if R.dim() == 3:
            self.n_refs = R.shape[0]
            if self.n_refs != max_epochs:
                raise DiaError("a 3-D reference stack needs max_epochs == R.shape[0]")
        self.n_rows, self.n_cols = R.shape[-2:]
        self.np = m * m + (bg_degree + 1) * (bg_degree + 2) // 2
        self.stream = stream
        self._h = dia_create(self.n_rows, self.n_cols, m, R, max_epochs=max_epochs, loss=loss,
                             huber_c=huber_c, noise=noise, sigma0=sigma0, gain=gain, d_flat=flat,
                             stream=stream, n_refs=self.n_refs, lambda_reg=lambda_reg, bg_degree=bg_degree)

    @property
    def raw(self) -> int:
        return self._h

    def info(self) -> dict:
        v = [C.c_int() for _ in range(4)]
        _check(load_library().dia_get_info(self._h, *[C.byref(x) for x in v]), self._h)
        return dict(grid_blocks=v[0].value, threads_per_block=v[1].value, smem_bytes=v[2].value,
                    launches_per_eval=v[3].value)

    def _epochs(self, I):
        return 1 if I.dim() == 2 else I.shape[0]

    def eval_loss_grad(self, I, theta, mask=None, var=None, loss=None, grad=None):
        """The outputs are allocated on, and written in the order of, the HANDLE's stream (`with` block below): a
        handle created with its own stream gives tensors that are safe to use on that stream; on any other
        stream synchronise first (Handle.synchronize())."""
        E = self._epochs(I)
        dev = I.device
        with self._stream_ctx():
            loss = torch.empty(E, dtype=torch.float64, device=dev) if loss is None else loss
            grad = torch.empty((E, self.np), dtype=torch.float64, device=dev) if grad is None else grad
            dia_eval_loss_grad(self._h, E, I, mask, var, theta, loss, grad)
        return loss, grad

    def synchronize(self):
        """Waits for everything enqueued on the handle's stream."""
        (self.stream if self.stream is not None else torch.cuda.current_stream(self.R.device)).synchronize()

    def difference_image(self, I, theta, mask=None, var=None):
        """-> (D float32 [E][n_rows][n_cols], metrics float64 [E][4] = N_used, MFB, MFV, chi^2), CUDA tensors."""
        E = self._epochs(I)
        with self._stream_ctx():
            D = torch.empty((E, self.n_rows, self.n_cols), dtype=torch.float32, device=I.device)
            metrics = torch.empty((E, 4), dtype=torch.float64, device=I.device)
            dia_difference_image(self._h, E, I, mask, var, theta, D, metrics)
        return D, metrics

    def hessian(self, I, theta, mask=None, var=None):
        """-> H float64 [np][np] CUDA tensor: Hessian of the objective at theta for the single target I."""
        with self._stream_ctx():
            H = torch.empty((self.np, self.np), dtype=torch.float64, device=I.device)
            dia_hessian(self._h, I, mask, var, theta, H)
        return H

    def covariance(self, H, want_cov: bool = True):
        """-> (cov float64 [np][np] or None, sigma float64 [np], info float64 [5]) CUDA tensors from the Hessian H
        (Eq. 16-17); info = (valid, ln det H, sigma_P, smallest Cholesky pivot, first non-positive pivot or -1)."""
        with self._stream_ctx():
            cov = torch.empty((self.np, self.np), dtype=torch.float64, device=H.device) if want_cov else None
            sigma = torch.empty(self.np, dtype=torch.float64, device=H.device)
            info = torch.empty(5, dtype=torch.float64, device=H.device)
            dia_covariance(self._h, H, cov, sigma, info)
        return cov, sigma, info

    def fit(self, I, theta0, opts: Optional[FitOpts] = None, mask=None, var=None):
        """Returns (theta_hat float32 [E][np] CUDA tensor, list[FitResult]); synchronises to read results."""
        E = self._epochs(I)
        opts = opts or FitOpts.default()
        with self._stream_ctx():                    # allocate, fit and read back in the order of the handle's stream
            theta = theta0.clone().reshape(E, self.np).contiguous()
            res = torch.zeros(E * C.sizeof(FitResult), dtype=torch.uint8, device=I.device)
            dia_fit(self._h, opts, E, I, mask, var, theta, res)
            host = res.cpu().numpy().tobytes()      # synchronises that stream
        out = [FitResult.from_buffer_copy(host[i * C.sizeof(FitResult):(i + 1) * C.sizeof(FitResult)])
               for i in range(E)]
        return theta, out

    # ---- host-buffer entry points: dia_fit_host / dia_eval_loss_grad_host of the C ABI (staging buffers, copy
    # stream and the chunked copy / fit overlap live in the library); only the pinned OUTPUT buffers are kept here
    def _host_out(self, E: int):
        if getattr(self, "_host_E", None) != E:
            self._host_E = E
            self._hres = torch.empty(E * C.sizeof(FitResult), dtype=torch.uint8).pin_memory()
            self._hth = torch.empty((E, self.np), dtype=torch.float32).pin_memory()
            self._hloss = torch.empty(E, dtype=torch.float64).pin_memory()
            self._hgrad = torch.empty((E, self.np), dtype=torch.float64).pin_memory()

    def _stream_ctx(self):
        """Context in which torch's current stream is the handle's stream.  A handle without a stream of its own
        runs on the legacy default stream like torch's default: nothing to switch (and no per-call cost -- a stream
        context costs several microseconds of host time, as much as a small evaluation).  A handle with its own
        stream first makes that stream wait for the caller's current stream, so inputs produced there are complete."""
        if self.stream is None:
            return _NO_CTX
        cur = torch.cuda.current_stream(self.R.device)
        if self.stream == cur:
            return _NO_CTX
        self.stream.wait_stream(cur)
        return torch.cuda.stream(self.stream)

    def fit_host(self, I_host: torch.Tensor, theta0_host: torch.Tensor, opts: Optional[FitOpts] = None,
                 mask_host: Optional[torch.Tensor] = None, chunks: Optional[int] = None):
        """dia_fit_host: dia_fit with HOST inputs and outputs (pinned tensors make the copies asynchronous).  The
        library copies I, theta0 (and the mask) to its staging buffers in `chunks` groups of epochs (default 4 when
        there are at least 8 epochs) on a second stream while the previous group is being fitted, copies theta-hat and
        the result structs back and synchronises.
        Returns (theta_hat [E][np] float32 host tensor, list[FitResult], bytes host->device, bytes device->host);
        theta_hat is a copy (the pinned output buffers are reused by the next call)."""
        E = 1 if I_host.dim() == 2 else I_host.shape[0]
        self._host_out(E)
        opts = opts or FitOpts.default()
        self._hth.copy_(theta0_host.reshape(E, self.np))            # in: theta0, out: theta-hat
        dia_fit_host(self._h, opts, E, I_host, mask_host, self._hth, self._hres, 0 if chunks is None else chunks)
        nres = C.sizeof(FitResult)
        raw = self._hres.numpy().tobytes()
        res = [FitResult.from_buffer_copy(raw[i * nres:(i + 1) * nres]) for i in range(E)]
        h2d = I_host.numel() * 4 + self._hth.numel() * 4 + (mask_host.numel() if mask_host is not None else 0)
        d2h = self._hth.numel() * 4 + self._hres.numel()
        return self._hth.clone(), res, h2d, d2h

    def eval_loss_grad_host(self, I_host: torch.Tensor, theta_host: torch.Tensor):
        """dia_eval_loss_grad_host: dia_eval_loss_grad with HOST inputs and outputs; returns (loss, grad, bytes h2d,
        bytes d2h); loss and grad are copies (the pinned output buffers are reused by the next call)."""
        E = 1 if I_host.dim() == 2 else I_host.shape[0]
        self._host_out(E)
        dia_eval_loss_grad_host(self._h, E, I_host, theta_host, self._hloss, self._hgrad)
        return (self._hloss.clone(), self._hgrad.clone(), I_host.numel() * 4 + theta_host.numel() * 4,
                self._hloss.numel() * 8 + self._hgrad.numel() * 8)

    def close(self):
        if self._h:
            dia_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
