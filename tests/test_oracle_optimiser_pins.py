"""External pins of the oracle's optimiser beyond its first step (no GPU).

The paper names the library for both phases -- Adam "as recommended in Kingma & Ba" and L-BFGS,
"the in-built algorithm" of the same library -- so the oracle's step-by-step restatement
(oracle/dia_ref_fit.c) is checked here against
  (a) `torch.optim.Adam` in float64 with two parameter groups, driven by the oracle's own (pinned) gradient,
  (b) the dense BFGS inverse-Hessian recursion H+ = (I - rho s y')H(I - rho y s') + rho s s' started from
      gamma I (Nocedal & Wright Eq. 6.17 / 7.20), written out in numpy -- the two-loop recursion of Alg. 7.4 must
      give the same direction,
  (c) the same with a history of 2, so that pairs are evicted,
  (d) the switch rule (reading R6: consecutive pre-update losses, strict <, denominator |L_{t-1}|) on tolerances
      crafted so that each alternative reading would switch at a different iteration.
`oracle.fit_trace` runs the same routine as `oracle.fit` and records the FP64 iterates.  None of the expected values
comes from the routine under test: they are rebuilt from the gradients at the recorded iterates.
"""
import numpy as np
import pytest

import oracle
from test_oracle_grad_fit import _dyadic_problem

torch = pytest.importorskip("torch")


def _quadratic(n=24, m=3, seed=21, noise=True):
    """FIXED-variance Gaussian objective: a strictly convex quadratic in theta."""
    R, I, th_true, _ = _dyadic_problem(n=n, m=m, seed=seed, noise=noise)
    var = (25.0 + I.clip(0)).astype(np.float32)
    cfg = oracle.RefConfig(n, n, m, noise=oracle.NOISE_FIXED)
    th0 = np.concatenate([np.full(m * m, 1.0 / (m * m)), [0.0]]).astype(np.float32)
    return cfg, R, I, var, th0


def _grad_at(cfg, R, I, var, theta64):
    """oracle gradient at the float32 rounding of theta (reading R9: theta is rounded where it enters the objective)"""
    L, g = oracle.eval_loss_grad(cfg, R, I, np.asarray(theta64, np.float64).astype(np.float32), var=var)
    return float(L[0]), g[0].copy()


# ------------------------------------------------------------------------------------------ (a) Adam
@pytest.mark.parametrize("lr_b0,noise_model", [(10.0, False), (1.0, True)])
def test_adam_trajectory_equals_torch_optim_adam(lr_b0, noise_model):
    """25 Adam updates (Eq. 9; K&B Alg. 1, R5) against torch.optim.Adam(float64) with the paper's two
    learning rates (kernel pixels 1e-3, B0 lr_b0).  A wrong bias correction, an epsilon inside the
    root, swapped betas, moments that are not carried over, or the wrong learning rate on B0 all show at t >= 2."""
    cfg, R, I, var, th0 = _quadratic()
    if noise_model:                      # Eq. 6 noise: the non-quadratic objective the fits really minimise
        cfg = oracle.RefConfig(cfg.n_rows, cfg.n_cols, cfg.m, sigma0=5.0, gain=1.0)
        var = None
    n_it = 25
    opts = oracle.RefFitOpts.default(force_adam_iters=n_it, force_lbfgs_iters=0, lr_b0=lr_b0)
    _, res, tr, trL = oracle.fit_trace(cfg, R, I, th0, opts, var=var)
    assert res.n_adam == n_it and res.n_lbfgs == 0 and tr.shape == (n_it, th0.size)

    nk = cfg.m * cfg.m
    pk = torch.tensor(th0[:nk].astype(np.float64), requires_grad=True)
    pb = torch.tensor(th0[nk:].astype(np.float64), requires_grad=True)
    opt = torch.optim.Adam([{"params": [pk], "lr": 1e-3}, {"params": [pb], "lr": lr_b0}],
                           betas=(0.9, 0.999), eps=1e-8, weight_decay=0.0, amsgrad=False)
    for t in range(n_it):
        theta = np.concatenate([pk.detach().numpy(), pb.detach().numpy()])
        L, g = _grad_at(cfg, R, I, var, theta)
        assert L == trL[t]                                   # the loss each update was computed from
        pk.grad = torch.from_numpy(g[:nk].copy())
        pb.grad = torch.from_numpy(g[nk:].copy())
        opt.step()
        theta = np.concatenate([pk.detach().numpy(), pb.detach().numpy()])
        err = np.abs(theta - tr[t]).max()
        assert err <= 1e-12 * max(1.0, np.abs(tr[t]).max()), (t, err)
    # the trajectory moved by many learning rates, so the comparison is not vacuous
    assert np.abs(tr[-1][:nk] - th0[:nk]).max() > 10 * 1e-3


# ------------------------------------------------------------------------------------------ (b), (c) L-BFGS
def _dense_lbfgs_direction(g, pairs):
    """-H g with H built by the BFGS inverse update over `pairs` (oldest first) from gamma I, gamma = s'y / y'y of
    the newest pair (N&W Eq. 7.20); gamma = 1 without pairs."""
    n = g.size
    if not pairs:
        return -g
    s, y = pairs[-1]
    H = (s @ y) / (y @ y) * np.eye(n)
    for s, y in pairs:
        rho = 1.0 / (y @ s)
        V = np.eye(n) - rho * np.outer(y, s)
        H = V.T @ H @ V + rho * np.outer(s, s)
    return -H @ g


@pytest.mark.parametrize("history,n_it", [(100, 7), (2, 7), (1, 5), (3, 9)])
def test_lbfgs_direction_equals_dense_bfgs_recursion(history, n_it):
    """Every L-BFGS step k of the oracle equals alpha_k * (-H_k g_k) with H_k the dense matrix built from the pairs
    the algorithm is supposed to hold at that point: all of them (history 100) or only the newest `history`
    (FIFO eviction).  alpha = 1, except the first step, scaled by min(1, 1/|g|_1) (R7).  A
    sign or order slip in either loop of Alg. 7.4, gamma taken from the wrong pair, rho = s'y instead of its
    inverse, or evicting the newest pair instead of the oldest all give O(1) deviations."""
    cfg, R, I, var, th0 = _quadratic(seed=22)
    # a few Adam steps first, so that L-BFGS starts away from the flat initial kernel
    opts = oracle.RefFitOpts.default(force_adam_iters=3, force_lbfgs_iters=n_it, lbfgs_history=history, lr_b0=1.0)
    _, res, tr, trL = oracle.fit_trace(cfg, R, I, th0, opts, var=var)
    assert res.n_adam == 3 and res.n_lbfgs == n_it and res.n_evals == 3 + 1 + n_it      # the switch re-uses its evaluation
    th = tr[2:]                                              # th[0] = start of L-BFGS, th[k+1] after step k
    grads = [_grad_at(cfg, R, I, var, t)[1] for t in th]
    pairs = []
    moved = 0.0
    for k in range(n_it):
        g = grads[k]
        held = pairs[-history:]
        d = _dense_lbfgs_direction(g, held)
        alpha = 1.0
        if not held:
            g1 = np.abs(g).sum()
            alpha = 1.0 / g1 if g1 > 1.0 else 1.0
        step = th[k + 1] - th[k]
        assert g @ d < 0
        err = np.abs(step - alpha * d).max()
        assert err <= 1e-8 * np.abs(alpha * d).max(), (k, err, np.abs(alpha * d).max())
        s, y = step, grads[k + 1] - g
        assert s @ y > 1e-10                                 # R7 curvature guard: every pair of this problem is kept
        pairs.append((s, y))
        moved = max(moved, np.abs(step).max())
        assert trL[3 + k] == _grad_at(cfg, R, I, var, th[k + 1])[0]
    assert moved > 1e-3
    if history < n_it - 1:                                   # eviction did happen and mattered
        d_all = _dense_lbfgs_direction(grads[n_it - 1], pairs[:n_it - 1])
        d_held = _dense_lbfgs_direction(grads[n_it - 1], pairs[:n_it - 1][-history:])
        assert np.abs(d_all - d_held).max() > 1e-6 * np.abs(d_held).max()


def test_lbfgs_full_history_terminates_on_quadratic_like_bfgs():
    """On a strictly convex quadratic with n parameters, BFGS with exact line searches terminates in n steps; with unit
    steps it does not, but the dense-recursion identity above implies the iterates converge to the normal-equation
    solution.  Checked here against numpy's least-squares solution of the same weighted problem (not the oracle's
    B08 routine): the end point of 60 L-BFGS steps."""
    cfg, R, I, var, th0 = _quadratic(seed=23)
    n, m, h = cfg.n_rows, cfg.m, (cfg.m - 1) // 2
    cols = [R.astype(np.float64)[a:n - 2 * h + a, b:n - 2 * h + b].ravel() for a in range(m) for b in range(m)]
    X = np.stack(cols + [np.ones_like(cols[0])], axis=1)
    sw = 1.0 / np.sqrt(var.astype(np.float64)[h:n - h, h:n - h].ravel())
    yv = I.astype(np.float64)[h:n - h, h:n - h].ravel()
    ls = np.linalg.lstsq(X * sw[:, None], yv * sw, rcond=None)[0]
    opts = oracle.RefFitOpts.default(force_adam_iters=0, force_lbfgs_iters=60)
    _, res, tr, _ = oracle.fit_trace(cfg, R, I, th0, opts, var=var)
    assert np.abs(tr[-1] - ls).max() <= 2e-5 * max(1.0, np.abs(ls).max())


# ------------------------------------------------------------------------------------------ (d) switch rule
def _first_switch(L, tol, strict=True, denom_prev=True):
    """t (1-based evaluation index) at which the Adam phase ends under the stated reading, given the losses
    L[0] = L_1, L[1] = L_2, ... at consecutive pre-update iterates."""
    for t in range(2, len(L) + 1):
        dL = abs(L[t - 1] - L[t - 2])
        ref = tol * abs(L[t - 2] if denom_prev else L[t - 1])
        if (dL < ref) if strict else (dL <= ref):
            return t
    return None


def test_switch_rule_strict_less_and_previous_loss_denominator():
    """"if between any two steepest descent updates the relative change in the loss is less than
    [tol] ... a L-BFGS optimiser takes over"; reading R6: losses at consecutive pre-update iterates, strict <,
    denominator |L_{t-1}|, L-BFGS starts from the iterate where the test fired and re-uses that evaluation."""
    cfg, R, I, var, th0 = _quadratic(seed=24)
    n_rec = 80
    opts = oracle.RefFitOpts.default(force_adam_iters=n_rec, force_lbfgs_iters=0, lr_b0=1.0)
    _, _, _, L = oracle.fit_trace(cfg, R, I, th0, opts, var=var)
    L = list(L)
    rel = [abs(L[t - 1] - L[t - 2]) / abs(L[t - 2]) for t in range(2, n_rec + 1)]       # rel[t-2] belongs to t

    def run(tol):
        o = oracle.RefFitOpts.default(tol_switch=tol, lr_b0=1.0, force_lbfgs_iters=0, max_adam_iters=n_rec - 2)
        _, res, _, _ = oracle.fit_trace(cfg, R, I, th0, o, var=var)
        return res

    # 1. "t >= 2": an enormous tolerance still needs two losses to compare -- one Adam update, two evaluations
    res = run(1e30)
    assert (res.n_adam, res.n_evals) == (1, 2)
    # 2. strict "<": a tolerance that makes |dL| == tol |L_{t-1}| exactly at some t* must not fire there
    found = False
    for ts in range(5, n_rec - 5):
        dL, Lp = abs(L[ts - 1] - L[ts - 2]), abs(L[ts - 2])
        tol = dL / Lp
        if tol * Lp != dL or _first_switch(L, tol, strict=False) != ts:
            continue
        expect = _first_switch(L, tol)
        assert expect is not None and expect != ts
        res = run(tol)
        assert res.n_adam == expect - 1 and res.n_evals == expect, (ts, expect, res.n_adam)
        found = True
        break
    assert found, "no iteration with an exactly representable tolerance -- change the seed"
    # 3. denominator |L_{t-1}|, not |L_t|: a tolerance between |dL|/|L_{t-1}| and |dL|/|L_t|
    found = False
    for ts in range(5, n_rec - 5):
        dL, Lp, Lt = abs(L[ts - 1] - L[ts - 2]), abs(L[ts - 2]), abs(L[ts - 1])
        lo, hi = dL / Lp, dL / Lt
        if not lo < hi:
            continue
        tol = 0.5 * (lo + hi)
        if _first_switch(L, tol) != ts or _first_switch(L, tol, denom_prev=False) == ts:
            continue
        res = run(tol)
        assert res.n_adam == ts - 1 and res.n_evals == ts
        found = True
        break
    assert found, "no discriminating iteration -- change the seed"
    # the recorded relative changes do fall through the paper's 1e-6 on this problem only much later: the tests above
    # are about the comparison, not about that value
    assert min(rel) < max(rel)


# ------------------------------------------------------------------------------------------ what is NOT pinned, and why
_SELF_CHECK = """
import json, sys
import numpy as np
import oracle
from workloads import make_workload
w = make_workload(1, n=160, m=9)
cfg = oracle.RefConfig(w.n, w.n, w.m, sigma0=w.sigma0, gain=w.gain)
th, r = oracle.fit(cfg, w.R, w.I, w.theta0)
print(json.dumps(dict(threads=oracle.num_threads(), n_adam=r[0].n_adam, n_lbfgs=r[0].n_lbfgs, status=r[0].status,
                      P=r[0].photometric_scale, loss=r[0].loss, theta=th[0].astype(float).tolist())))
"""


def test_stopped_iterate_depends_on_summation_order():
    """Why the stopped iterate of a free-running fit is "parity unpinned": the oracle itself does
    not reproduce it.  The same fit (config 1 at 160^2, 9x9 kernel, paper settings) with 3 and with 4 OpenMP threads --
    two orders of the same FP64 sums, 1e-16 apart -- stops after different numbers of L-BFGS iterations and its
    kernels differ by far more than north_star's 1e-4, while the photometric scale and the loss (what the data
    determine) agree.  No implementation, in any precision, can match such an iterate to 1e-4; the fit-parity
    protocol therefore asserts lock-step and well-conditioned (converged / regularised) fits strictly and the
    stopped iterate through the model image."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    runs = []
    for threads in (3, 4):
        env = dict(os.environ, OMP_NUM_THREADS=str(threads), PYTHONPATH=root)
        out = subprocess.run([sys.executable, "-c", _SELF_CHECK], env=env, cwd=root, capture_output=True, text=True, check=True)
        runs.append(json.loads(out.stdout.strip().splitlines()[-1]))
    a, b = runs
    assert (a["threads"], b["threads"]) == (3, 4)
    assert a["status"] in (0, 1) and b["status"] in (0, 1)
    assert a["n_adam"] == b["n_adam"]                       # the Adam phase is robust at this horizon ...
    Ka, Kb = np.array(a["theta"][:-1]), np.array(b["theta"][:-1])
    dK = np.abs(Ka - Kb).max() / np.abs(Ka).max()
    dP = abs(a["P"] - b["P"]) / abs(a["P"])
    dL = abs(a["loss"] - b["loss"]) / abs(a["loss"])
    print(f"oracle vs oracle (3 / 4 threads): lbfgs {a['n_lbfgs']} / {b['n_lbfgs']}, dK={dK:.2e} dP={dP:.2e} dL={dL:.2e}")
    assert a["n_lbfgs"] != b["n_lbfgs"]                     # ... the stop rule fires at different L-BFGS iterations
    assert dK > 10 * 1e-4                                   # the kernels differ by far more than the parity tolerance
    assert dP <= 1e-4 and dL <= 1e-4                        # the scale factor and the loss do not
