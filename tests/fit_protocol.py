"""Fit-parity protocol of SURVEY.md 8(c.6) / DESIGN.md section 6, shared by the GPU fit tests (not a test module).

free-running fit, same theta_init and options on both sides:
  strict criterion   |dP| <= 1e-4 |P|,  |dB0| <= 1e-4 max(|B0|, 1),  max|dK| <= 1e-4 max|K_or|
  reported with it   |dL|/|L|, iteration counts and status on both sides, cond(H) at the oracle's theta-hat, and the
                     conditioning-aware norms
                         e_H = sqrt(dtheta' H dtheta / theta' H theta)        (H: the oracle's Hessian at its theta-hat)
                         e_M = |R (x) dK + dB0|_2 / |M|_2                      (difference of the two model images)
  lock-step re-run   when only the K criterion fails: the device repeats the fit with force_*_iters = the oracle's
                     counts and is compared again.
Everything here calls the oracle and numpy only; the device results are passed in.
"""
from __future__ import annotations

import dataclasses

import numpy as np

import oracle

TOL = 1e-4


@dataclasses.dataclass
class FitDiff:
    dK: float
    dP: float
    dB0: float
    dL: float
    e_H: float = float("nan")
    e_M: float = float("nan")
    cond: float = float("nan")

    @property
    def strict(self) -> bool:
        return self.dK <= TOL and self.dP <= TOL and self.dB0 <= TOL

    @property
    def only_K_fails(self) -> bool:
        return self.dK > TOL and self.dP <= TOL and self.dB0 <= TOL


def diff(cfg, tho, ro, thg, rg) -> FitDiff:
    """theta [np] of one epoch from the oracle (tho, ro) and the device (thg, rg)."""
    nk = cfg.m * cfg.m
    Ko, Kg = tho[:nk].astype(np.float64), thg[:nk].astype(np.float64)
    dK = float(np.abs(Kg - Ko).max() / np.abs(Ko).max())
    dP = abs(rg.photometric_scale - ro.photometric_scale) / abs(ro.photometric_scale)
    dB0 = abs(float(thg[nk]) - float(tho[nk])) / max(abs(float(tho[nk])), 1.0)
    dL = abs(rg.loss - ro.loss) / abs(ro.loss) if ro.loss != 0 else abs(rg.loss)
    return FitDiff(dK, dP, dB0, dL)


def conditioning(cfg, R, I, tho, thg, d: FitDiff, mask=None, var=None, H=None):
    """Fills cond(H) and the conditioning-aware norms; H defaults to the oracle's Hessian at its own theta-hat
    (O(n^2 m^4): only at sizes where that takes seconds -- pass a Hessian from elsewhere otherwise)."""
    if H is None:
        H = oracle.hessian(cfg, R, I, np.asarray(tho, np.float32), mask=mask, var=var)
    ev = np.linalg.eigvalsh(H)
    d.cond = float(ev[-1] / ev[0]) if ev[0] > 0 else float("inf")
    to, dt = tho.astype(np.float64), thg.astype(np.float64) - tho.astype(np.float64)
    d.e_H = float(np.sqrt(max(dt @ H @ dt, 0.0) / (to @ H @ to)))
    plain = oracle.RefConfig(cfg.n_rows, cfg.n_cols, cfg.m, bg_degree=cfg.bg_degree)
    Mo = oracle.model(plain, R, np.asarray(tho, np.float32))
    dM = oracle.model(plain, R, np.asarray(dt, np.float32))       # the model is linear in theta: R (x) dK + dB0
    d.e_M = float(np.linalg.norm(dM) / np.linalg.norm(Mo))
    return H


def report(tag, e, d: FitDiff, ro, rg) -> str:
    line = (f"{tag} e{e}: dK={d.dK:.2e} dP={d.dP:.2e} dB0={d.dB0:.2e} dL={d.dL:.2e} e_H={d.e_H:.2e} e_M={d.e_M:.2e} "
            f"cond(H)={d.cond:.2e} | device adam={rg.n_adam} lbfgs={rg.n_lbfgs} evals={rg.n_evals} st={rg.status} "
            f"|g|={rg.grad_inf_norm:.2e} | oracle adam={ro.n_adam} lbfgs={ro.n_lbfgs} evals={ro.n_evals} st={ro.status} "
            f"|g|={ro.grad_inf_norm:.2e} | strict={'yes' if d.strict else 'NO'}")
    print(line, flush=True)
    return line
