"""Pins of the oracle's gradient, B08 solve and optimiser (no GPU)."""
import math

import numpy as np
import pytest
import scipy.signal

import oracle
from workloads import make_workload, n_valid


def _dyadic_problem(n=14, m=3, seed=3, noise=True):
    """theta and steps exactly representable in float32, so finite differences of the
    float32-theta objective are exact in the argument."""
    rng = np.random.default_rng(seed)
    R = (60.0 + np.floor(400.0 * rng.random((n, n)) ** 4)).astype(np.float32)
    K = np.round(rng.random((m, m)) / (m * m) * 2 * 4096) / 4096
    th = np.concatenate([K.ravel(), [2.75]]).astype(np.float32)
    Mfull = R.astype(np.float64) * K.sum() + 2.75
    h = (m - 1) // 2
    Mfull[h:n - h, h:n - h] = scipy.signal.correlate2d(R.astype(np.float64), K, mode="valid") + 2.75
    I = Mfull + (rng.normal(0, 1, (n, n)) * np.sqrt(25 + Mfull) if noise else 0.0)
    flat = (0.9 + 0.2 * rng.random((n, n))).astype(np.float32)
    return R, I.astype(np.float32), th, flat


def _fd_grad(cfg, R, I, th, mask=None, var=None):
    """Richardson-extrapolated central differences with steps that are exact in float32
    (2^-18, 2^-17 for kernel pixels, 2^-11, 2^-10 for B0): small enough that almost no pixel
    crosses the Huber kink |z| = c inside a step."""
    g = np.zeros(th.size)
    for k in range(th.size):
        d = []
        for hstep in ((2.0 ** -18, 2.0 ** -17) if k < th.size - 1 else (2.0 ** -11, 2.0 ** -10)):
            tp, tm = th.copy(), th.copy()
            tp[k] += np.float32(hstep)
            tm[k] -= np.float32(hstep)
            assert float(tp[k]) - float(tm[k]) == 2 * hstep
            Lp, _ = oracle.eval_loss_grad(cfg, R, I, tp, mask=mask, var=var)
            Lm, _ = oracle.eval_loss_grad(cfg, R, I, tm, mask=mask, var=var)
            d.append((Lp[0] - Lm[0]) / (2 * hstep))
        g[k] = (4 * d[0] - d[1]) / 3
    return g


@pytest.mark.parametrize("loss", [oracle.LOSS_GAUSSIAN, oracle.LOSS_HUBER])
@pytest.mark.parametrize("noise_mode", [oracle.NOISE_MODEL, oracle.NOISE_FIXED])
def test_gradient_vs_finite_differences(loss, noise_mode):
    """D1: w = -psi/s - psi z b'/(2v) + b'/(2v).  The paper prints no gradient
    (autodiff), so the derived formula is checked against central differences
    of the oracle's own loss, which the closed-form tests pin.  Catches a dropped term, a
    wrong sign, a transposed R index in g_K and a missing flat/gain factor."""
    R, I, th, flat = _dyadic_problem()
    n, m = R.shape[0], 3
    I = I.copy()
    I[5, 6] += 400.0                                    # one outlier => Huber linear branch
    var = (20.0 + 0.5 * I.clip(0)).astype(np.float32) if noise_mode == oracle.NOISE_FIXED else None
    cfg = oracle.RefConfig(n, n, m, loss=loss, huber_c=1.345, noise=noise_mode, sigma0=5.0,
                           gain=1.6, flat=flat)
    mask = np.ones((n, n), np.uint8)
    mask[3, 4] = 0
    L, g = oracle.eval_loss_grad(cfg, R, I, th, mask=mask, var=var)
    fd = _fd_grad(cfg, R, I, th, mask=mask, var=var)
    scale = np.abs(g[0]).max()
    assert np.abs(g[0] - fd).max() <= 2e-7 * scale


def test_gradient_vs_torch_autograd():
    """Same check by the paper's own route: float64 autograd through conv2d of Eq. 8 with
    Eq. 6."""
    torch = pytest.importorskip("torch")
    R, I, th, flat = _dyadic_problem(n=16, m=5, seed=8)
    n, m, h = 16, 5, 2
    s0, G = 4.0, 2.0
    cfg = oracle.RefConfig(n, n, m, sigma0=s0, gain=G, flat=flat)
    L, g = oracle.eval_loss_grad(cfg, R, I, th)
    K = torch.tensor(th[:-1].astype(np.float64).reshape(1, 1, m, m), requires_grad=True)
    B0 = torch.tensor(float(th[-1]), dtype=torch.float64, requires_grad=True)
    Rt = torch.from_numpy(R.astype(np.float64))[None, None]
    M = torch.nn.functional.conv2d(Rt, K)[0, 0] + B0
    Fv = torch.from_numpy(flat.astype(np.float64))[h:n - h, h:n - h]
    Iv = torch.from_numpy(I.astype(np.float64))[h:n - h, h:n - h]
    var = s0 ** 2 / Fv ** 2 + M / (G * Fv)
    loss = 0.5 * ((Iv - M) ** 2 / var).sum() + torch.log(torch.sqrt(var)).sum()
    loss.backward()
    assert L[0] == pytest.approx(loss.item(), rel=1e-13)
    ref = np.concatenate([K.grad.numpy().ravel(), [B0.grad.item()]])
    assert np.abs(g[0] - ref).max() <= 1e-12 * np.abs(ref).max()


def test_model_mode_gradient_at_zero_residual_D2():
    """D2: at r = 0 in MODEL mode w = b/(2v), so g_p = sum_V X_p / (2 G F v) -- the log-sigma
    term alone.  This is why noise-free MODEL fits sit at B0_true - 1/(2G) (R12)."""
    R, I, th, flat = _dyadic_problem(noise=False)
    n, m, h = R.shape[0], 3, 1
    G, s0 = 2.0, 5.0
    cfg = oracle.RefConfig(n, n, m, sigma0=s0, gain=G, flat=flat)
    M = oracle.model(cfg, R, th)
    assert np.array_equal(M.astype(np.float32).astype(np.float64), M)      # dyadic: I == M exactly
    L, g = oracle.eval_loss_grad(cfg, R, I, th)
    F = flat.astype(np.float64)[h:n - h, h:n - h]
    v = s0 ** 2 / F ** 2 + M / (G * F)
    w = 1.0 / (2 * G * F * v)
    assert L[0] == pytest.approx(0.5 * np.log(v).sum(), rel=1e-13)
    assert g[0][-1] == pytest.approx(w.sum(), rel=1e-12)
    for a in range(m):
        for b in range(m):
            X = R.astype(np.float64)[a:a + n - m + 1, b:b + n - m + 1]
            assert g[0][a * m + b] == pytest.approx((w * X).sum(), rel=1e-12)


def test_mask_and_border_poison():
    """R4: a masked pixel contributes nothing; pixels of I outside the valid set are never read."""
    R, I, th, flat = _dyadic_problem()
    n, m, h = R.shape[0], 3, 1
    cfg = oracle.RefConfig(n, n, m, sigma0=5.0, gain=1.0)
    L0, g0 = oracle.eval_loss_grad(cfg, R, I, th)
    Ip = I.copy()
    Ip[:h, :] = np.nan; Ip[-h:, :] = np.nan; Ip[:, :h] = np.nan; Ip[:, -h:] = np.nan
    L1, g1 = oracle.eval_loss_grad(cfg, R, Ip, th)
    assert L0[0] == L1[0] and np.array_equal(g0, g1)
    # keep a single pixel: the result is that pixel's closed-form term with M from scipy
    mask = np.zeros((n, n), np.uint8)
    mask[6, 9] = 1
    L, g = oracle.eval_loss_grad(cfg, R, I, th, mask=mask)
    K = th[:-1].astype(np.float64).reshape(m, m)
    M = scipy.signal.correlate2d(R.astype(np.float64), K, mode="valid")[6 - h, 9 - h] + float(th[-1])
    v = 25.0 + M
    r = float(I[6, 9]) - M
    assert L[0] == pytest.approx(0.5 * r * r / v + 0.5 * math.log(v), rel=1e-13)
    w = -r / v - r * r / (2 * v * v) + 1 / (2 * v)
    assert g[0][-1] == pytest.approx(w, rel=1e-12)
    assert g[0][0 * m + 2] == pytest.approx(w * float(R[6 - h + 0, 9 - h + 2]), rel=1e-12)
    # masking removes exactly that term
    mask = 1 - mask
    L2, g2 = oracle.eval_loss_grad(cfg, R, I, th, mask=mask)
    assert L2[0] + L[0] == pytest.approx(L0[0], rel=1e-13)
    assert np.allclose(g2 + g, g0, rtol=1e-11, atol=1e-9)


def test_batched_epochs_equal_singles():
    w = make_workload(4, n=48, n_epochs=3, m=5)
    cfg = oracle.RefConfig(48, 48, 5, sigma0=w.sigma0, gain=w.gain)
    L, g = oracle.eval_loss_grad(cfg, w.R, w.I, w.theta0)
    for e in range(3):
        Le, ge = oracle.eval_loss_grad(cfg, w.R, w.I[e], w.theta0[e])
        assert Le[0] == L[e] and np.array_equal(ge[0], g[e])


# ---------------------------------------------------------------- B08 normal equations
def _design(R, m):
    n = R.shape[0]
    nv = n - m + 1
    cols = [R.astype(np.float64)[a:a + nv, b:b + nv].ravel() for a in range(m) for b in range(m)]
    cols.append(np.ones(nv * nv))
    return np.stack(cols, axis=1)


def test_b08_solve_vs_weighted_lstsq():
    """One B08 iteration with a given variance map is weighted linear least squares
    (PAPER.md:81); numpy's lstsq on the explicit design matrix is the library special case."""
    R, I, th, flat = _dyadic_problem(n=16, m=3, seed=5)
    n, m, h = 16, 3, 1
    var = (30.0 + 0.7 * I.clip(0)).astype(np.float32)
    cfg = oracle.RefConfig(n, n, m, noise=oracle.NOISE_FIXED)
    theta, H = oracle.b08_solve(cfg, R, I, var_fixed=var, n_iters=1, want_H=True)
    X = _design(R, m)
    sw = 1.0 / np.sqrt(var.astype(np.float64)[h:n - h, h:n - h].ravel())
    y = I.astype(np.float64)[h:n - h, h:n - h].ravel()
    ref, *_ = np.linalg.lstsq(X * sw[:, None], y * sw, rcond=None)
    assert np.allclose(theta, ref, rtol=1e-8, atol=1e-10)
    assert np.allclose(H, (X * sw[:, None]).T @ (X * sw[:, None]), rtol=1e-12)
    # FIXED + Gaussian gradient is H theta - rhs  (DESIGN.md c.5)
    t32 = th
    L, g = oracle.eval_loss_grad(cfg, R, I, t32, var=var)
    rhs = (X * (sw ** 2)[:, None]).T @ y
    assert np.allclose(g[0], H @ t32.astype(np.float64) - rhs, rtol=1e-9, atol=1e-8 * np.abs(g).max())
    # L_min = (sum I^2/v - rhs' theta_hat)/2
    th_hat32 = theta.astype(np.float32)
    Lmin, _ = oracle.eval_loss_grad(cfg, R, I, th_hat32, var=var)
    assert Lmin[0] == pytest.approx(0.5 * ((y * sw) ** 2).sum() - 0.5 * rhs @ theta, rel=1e-5)


def test_b08_three_iterations_recover_planted_noisy():
    """Iterated solve (sigma from the previous model) on config-0-like data lands
    within a few standard errors of the planted parameters; P = sum K (Eq. 3)."""
    w = make_workload(0, n=64, m=5)
    cfg = oracle.RefConfig(64, 64, 5, sigma0=w.sigma0, gain=w.gain)
    theta, H = oracle.b08_solve(cfg, w.R, w.I[0], n_iters=3, want_H=True)
    cov = np.linalg.inv(H)
    err = (theta - w.theta_true[0]) / np.sqrt(np.diag(cov))
    assert np.abs(err).max() < 5.0
    ones = np.concatenate([np.ones(25), [0.0]])
    sigP = math.sqrt(ones @ cov @ ones)
    assert abs(theta[:-1].sum() - 1.2) < 5 * sigP


# ---------------------------------------------------------------- optimiser
def test_adam_first_step_has_magnitude_lr():
    """Bias-corrected Adam at t = 1 moves every coordinate by lr_p * g/(|g| + eps)
    (Kingma & Ba Alg. 1; PAPER.md:242 per-parameter learning rates)."""
    w = make_workload(0, n=48, m=5)
    cfg = oracle.RefConfig(48, 48, 5, sigma0=w.sigma0, gain=w.gain)
    opts = oracle.RefFitOpts.default(force_adam_iters=1, force_lbfgs_iters=0, lr_b0=10.0)
    _, g = oracle.eval_loss_grad(cfg, w.R, w.I, w.theta0)
    th, res = oracle.fit(cfg, w.R, w.I, w.theta0, opts)
    step = th[0].astype(np.float64) - w.theta0[0].astype(np.float64)
    assert np.allclose(step[:-1], -1e-3 * np.sign(g[0][:-1]), rtol=1e-4)
    assert step[-1] == pytest.approx(-10.0 * np.sign(g[0][-1]), rel=1e-5)
    assert res[0].n_adam == 1 and res[0].n_lbfgs == 0 and res[0].n_evals == 2


def test_fit_fixed_weights_reaches_normal_equation_solution():
    """Noise-free target, FIXED variance: the objective is a strictly convex quadratic whose
    minimiser is the normal-equation solution = theta_true (PAPER.md:135 convexity; test (ii)
    of PAPER.md:453 in spirit).  Adam -> L-BFGS must land on it and P-hat on the planted scale."""
    R, I, th_true, _ = _dyadic_problem(n=24, m=3, seed=11, noise=False)
    n, m = 24, 3
    var = np.full((n, n), 25.0, np.float32)
    cfg = oracle.RefConfig(n, n, m, noise=oracle.NOISE_FIXED)
    ne = oracle.b08_solve(cfg, R, I, var_fixed=var, n_iters=1)
    assert np.allclose(ne, th_true.astype(np.float64), rtol=0, atol=1e-9)      # planted recovery
    th0 = np.concatenate([np.full(m * m, 1.0 / (m * m)), [0.0]]).astype(np.float32)
    opts = oracle.RefFitOpts.default(lr_b0=1.0, tol_change_rel=1e-14, tol_grad_abs=1e-9,
                                     max_lbfgs_iters=300)
    th, res = oracle.fit(cfg, R, I, th0, opts, var=var)
    P_true = float(th_true[:-1].astype(np.float64).sum())
    assert res[0].photometric_scale == pytest.approx(P_true, rel=2e-6)
    assert np.abs(th[0][:-1] - th_true[:-1]).max() < 2e-6
    assert abs(th[0][-1] - th_true[-1]) < 2e-4
    assert res[0].loss < 1e-6


def test_lbfgs_full_history_solves_quadratic():
    """L-BFGS alone (no Adam steps) on the same quadratic reaches the normal-equation solution
    (N&W Alg. 7.4/7.5)."""
    R, I, th_true, _ = _dyadic_problem(n=24, m=3, seed=12, noise=True)
    n, m = 24, 3
    var = (25.0 + I.clip(0)).astype(np.float32)
    cfg = oracle.RefConfig(n, n, m, noise=oracle.NOISE_FIXED)
    ne = oracle.b08_solve(cfg, R, I, var_fixed=var, n_iters=1)
    th0 = np.concatenate([np.full(m * m, 1.0 / (m * m)), [0.0]]).astype(np.float32)
    opts = oracle.RefFitOpts.default(force_adam_iters=0, tol_change_rel=1e-15, tol_grad_abs=1e-8,
                                     max_lbfgs_iters=400)
    th, res = oracle.fit(cfg, R, I, th0, opts, var=var)
    assert res[0].n_adam == 0
    Lne, _ = oracle.eval_loss_grad(cfg, R, I, ne.astype(np.float32), var=var)
    assert res[0].loss == pytest.approx(Lne[0], rel=1e-7)
    assert np.abs(th[0] - ne).max() < 5e-4 * max(1.0, np.abs(ne).max())


def test_noisy_fit_statistics_mfv(golden):
    """Eq. 29-30: after an unregularised fit MFB ~ 0 and
    MFV ~ 1 - (m^2+1)/N_valid < 1 (overfit by the parameter count; Table 2 prints 0.979 at
    142^2, m = 19 where 1 - 362/15376 = 0.976)."""
    assert abs((1 - 362 / 15376) - golden["table2_mfv_snr1_oversampled"]) < 0.01
    w = make_workload(0, n=96, m=7)
    cfg = oracle.RefConfig(96, 96, 7, sigma0=w.sigma0, gain=w.gain)
    th, res = oracle.fit(cfg, w.R, w.I, w.theta0)
    assert res[0].status in (0, 1)
    M = oracle.model(cfg, w.R, th[0])
    h = 3
    Mtrue = oracle.model(cfg, w.R, w.theta_true[0].astype(np.float32))
    sig = np.sqrt(w.sigma0 ** 2 + Mtrue)
    eps = (w.I[0].astype(np.float64)[h:-h, h:-h] - M) / sig
    N = n_valid(96, 7)
    assert abs(eps.mean()) < 4 / math.sqrt(N)
    mfv = eps.var(ddof=1)
    assert abs(mfv - (1 - 50 / N)) < 4 * math.sqrt(2 / N)
    assert res[0].photometric_scale == pytest.approx(1.2, abs=0.02)


# ---------------------------------------------------------------- Hessian (Eq. 15-17)
@pytest.mark.parametrize("loss", [oracle.LOSS_GAUSSIAN, oracle.LOSS_HUBER])
@pytest.mark.parametrize("noise_mode", [oracle.NOISE_MODEL, oracle.NOISE_FIXED])
def test_hessian_vs_finite_differences_of_gradient(loss, noise_mode):
    """D3: h = d^2 l/dM^2.  The paper takes the Hessian by autodiff, so the
    derived closed form is checked against central differences of the oracle's gradient, itself pinned
    above.  Catches a dropped or mis-signed term of dw/dM, a missing symmetrisation and a wrong
    background-block index."""
    R, I, th, flat = _dyadic_problem()
    n, m = R.shape[0], 3
    I = I.copy()
    I[5, 6] += 400.0
    var = (20.0 + 0.5 * I.clip(0)).astype(np.float32) if noise_mode == oracle.NOISE_FIXED else None
    cfg = oracle.RefConfig(n, n, m, loss=loss, huber_c=1.345, noise=noise_mode, sigma0=5.0, gain=1.6,
                           flat=flat, bg_degree=1, lambda_reg=0.3)
    th = np.concatenate([th, [0.5, -0.25]]).astype(np.float32)
    H = oracle.hessian(cfg, R, I, th, var=var)
    assert np.array_equal(H, H.T)
    fd = np.zeros_like(H)
    for k in range(th.size):
        step = 2.0 ** -16 if k < m * m else 2.0 ** -9
        tp, tm = th.copy(), th.copy()
        tp[k] += np.float32(step)
        tm[k] -= np.float32(step)
        assert float(tp[k]) - float(tm[k]) == 2 * step
        _, gp = oracle.eval_loss_grad(cfg, R, I, tp, var=var)
        _, gm = oracle.eval_loss_grad(cfg, R, I, tm, var=var)
        fd[:, k] = (gp[0] - gm[0]) / (2 * step)
    d = np.sqrt(np.abs(np.diag(H)))
    assert np.abs((H - fd) / np.outer(d, d)).max() < 1e-6


def test_hessian_vs_torch_autograd():
    """The paper's own route: float64 autograd Hessian of Eq. 8 with Eq. 6."""
    torch = pytest.importorskip("torch")
    R, I, th, flat = _dyadic_problem(n=12, m=3, seed=5)
    n, m, h = 12, 3, 1
    s0, G = 4.0, 2.0
    cfg = oracle.RefConfig(n, n, m, sigma0=s0, gain=G, flat=flat)
    H = oracle.hessian(cfg, R, I, th)
    Rt = torch.from_numpy(R.astype(np.float64))[None, None]
    Fv = torch.from_numpy(flat.astype(np.float64))[h:n - h, h:n - h]
    Iv = torch.from_numpy(I.astype(np.float64))[h:n - h, h:n - h]

    def f(t):
        M = torch.nn.functional.conv2d(Rt, t[:-1].reshape(1, 1, m, m))[0, 0] + t[-1]
        var = s0 ** 2 / Fv ** 2 + M / (G * Fv)
        return 0.5 * ((Iv - M) ** 2 / var).sum() + 0.5 * torch.log(var).sum()

    ref = torch.autograd.functional.hessian(f, torch.tensor(th.astype(np.float64))).numpy()
    assert np.abs(H - ref).max() <= 1e-11 * np.abs(ref).max()


def test_hessian_fixed_weights_is_normal_matrix():
    """FIXED noise, Gaussian loss: H = X' diag(1/var) X, the B08 normal matrix;
    its inverse is the textbook weighted-least-squares covariance (Eq. 16-17)."""
    R, I, th, _ = _dyadic_problem(n=18, m=5, seed=9)
    var = (30.0 + 0.4 * I.clip(0)).astype(np.float32)
    cfg = oracle.RefConfig(18, 18, 5, noise=oracle.NOISE_FIXED)
    H = oracle.hessian(cfg, R, I, th, var=var)
    X = _design(R, 5)
    wv = 1.0 / var.astype(np.float64)[2:-2, 2:-2].ravel()
    ref = X.T @ (X * wv[:, None])
    assert np.abs(H - ref).max() <= 1e-12 * np.abs(ref).max()
