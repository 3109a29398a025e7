"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Each test names the plausible mistake it is chosen to catch.  None of the expected values
comes from oracle/ itself or from the CUDA path: they are paper-printed values, closed forms,
library routines (scipy / torch float64) or brute force on tiny inputs.
"""
import math

import numpy as np
import pytest
import scipy.integrate
import scipy.signal

import oracle
from workloads import n_valid

RNG = np.random.default_rng(1234)


def _cfg(n, m, **kw):
    return oracle.RefConfig(n, n, m, **kw)


def _rand_problem(n=12, m=3, seed=0, sky=80.0):
    rng = np.random.default_rng(seed)
    R = (sky + 200.0 * rng.random((n, n)) ** 3).astype(np.float32)
    K = rng.random((m, m))
    K = 0.9 * K / K.sum()
    theta = np.concatenate([K.ravel(), [3.0]]).astype(np.float32)
    I = (R * 0.9 + 3.0 + rng.normal(0, 9.0, (n, n))).astype(np.float32)
    return R, I, theta


# ---------------------------------------------------------------- valid region
def test_n_data_paper_value(golden):
    """PAPER.md:365 prints N_data = 15376 for 142^2 images and a 19x19 kernel."""
    n, m = int(golden["n_data_image_size"]), int(golden["n_data_kernel_size"])
    assert n_valid(n, m) == int(golden["n_data_value"])
    R = np.ones((n, n), np.float32)
    th = np.zeros(m * m + 1, np.float32)
    assert oracle.model(_cfg(n, m), R, th).size == int(golden["n_data_value"])
    # every valid pixel contributes exactly once: with K = 0, B0 = 0, FIXED var = 1, I = 1
    # the loss is N_data * 1/2 (catches an off-by-one in the loop bounds)
    L, g = oracle.eval_loss_grad(_cfg(n, m, noise=oracle.NOISE_FIXED), R, R, th, var=R)
    assert L[0] == 0.5 * golden["n_data_value"]


# ---------------------------------------------------------------- model image, Eq. 2
def test_model_delta_and_shift_convention():
    """K = centred delta => M = crop(R) + B0 exactly.  Paper test (iii): a target
    equal to the reference shifted by +1 px in x and y is matched by a delta at kernel
    coordinates (l, m) = (-1, -1).  Catches a flipped kernel (convolution instead of the
    cross-correlation Eq. 2 prints) and swapped row/column offsets."""
    n, m, h = 16, 5, 2
    R = RNG.random((n, n)).astype(np.float32) * 100
    th = np.zeros(m * m + 1, np.float32)
    th[h * m + h] = 1.0
    th[-1] = 2.5
    M = oracle.model(_cfg(n, m), R, th)
    assert np.array_equal(M, R[h:n - h, h:n - h].astype(np.float64) + 2.5)
    # I_ij = R_(i-1)(j-1)  (content moved by +1 in each direction)
    I = np.roll(np.roll(R, 1, axis=0), 1, axis=1)
    th = np.zeros(m * m + 1, np.float32)
    th[(h - 1) * m + (h - 1)] = 1.0          # (l, mm) = (-1, -1)
    M = oracle.model(_cfg(n, m), R, th)
    assert np.array_equal(M, I[h:n - h, h:n - h].astype(np.float64))
    # asymmetric: a delta at (l, mm) = (+1, -2) picks R_(i+1)(j-2): rows and columns not swapped
    th = np.zeros(m * m + 1, np.float32)
    th[(h + 1) * m + (h - 2)] = 1.0
    M = oracle.model(_cfg(n, m), R, th)
    assert np.array_equal(M, R[h + 1:n - h + 1, h - 2:n - h - 2].astype(np.float64))


def test_model_constant_reference_and_library_correlation():
    """R == const => M = const * P + B0 (Eq. 3 link); general case against scipy's
    correlate2d and torch's float64 conv2d (the paper's own route)."""
    n, m = 20, 7
    R = np.full((n, n), 3.0, np.float32)
    K = RNG.random((m, m))
    th = np.concatenate([K.ravel(), [-4.0]]).astype(np.float32)
    P = th[:-1].astype(np.float64).sum()
    M = oracle.model(_cfg(n, m), R, th)
    assert np.allclose(M, 3.0 * P - 4.0, rtol=1e-14)
    R = (RNG.random((n, n)) * 1000).astype(np.float32)
    M = oracle.model(_cfg(n, m), R, th)
    K32 = th[:-1].reshape(m, m).astype(np.float64)
    ref = scipy.signal.correlate2d(R.astype(np.float64), K32, mode="valid") - 4.0
    assert np.allclose(M, ref, rtol=1e-13, atol=1e-10)
    torch = pytest.importorskip("torch")
    t = torch.nn.functional.conv2d(torch.from_numpy(R.astype(np.float64))[None, None],
                                   torch.from_numpy(K32)[None, None]).numpy()[0, 0] - 4.0
    assert np.allclose(M, t, rtol=1e-13, atol=1e-10)


def test_model_rectangular_image():
    n_r, n_c, m = 9, 14, 3
    R = (RNG.random((n_r, n_c)) * 50).astype(np.float32)
    th = RNG.random(m * m + 1).astype(np.float32)
    cfg = oracle.RefConfig(n_r, n_c, m)
    M = oracle.model(cfg, R, th)
    ref = scipy.signal.correlate2d(R.astype(np.float64), th[:-1].reshape(m, m).astype(np.float64),
                                   mode="valid") + np.float64(th[-1])
    assert M.shape == (n_r - 2, n_c - 2)
    assert np.allclose(M, ref, rtol=1e-13)


# ---------------------------------------------------------------- single-pixel closed forms
def _single_pixel(I, Rv, K, B0, **kw):
    """1x1 image, 1x1 kernel: the whole objective is one term."""
    cfg = oracle.RefConfig(1, 1, 1, **kw)
    L, g = oracle.eval_loss_grad(cfg, np.array([[Rv]], np.float32), np.array([[I]], np.float32),
                                 np.array([K, B0], np.float32),
                                 var=None if kw.get("noise", 0) == 0 else np.array([[kw.pop("_var", 1.0)]], np.float32))
    return L[0], g[0]


def test_gaussian_single_pixel_closed_form():
    """Eq. 8 with Eq. 6 at F = G = 1: v = sigma0^2 + M (the form of Eq. 22/25);
    L = r^2/(2v) + ln(v)/2.  Catches a missing 1/2, ln(sigma) vs ln(v), sigma vs sigma^2."""
    I, Rv, K, B0, s0 = 130.0, 100.0, 1.25, 2.0, 5.0
    M = K * Rv + B0
    v = s0 ** 2 + M
    L, g = _single_pixel(I, Rv, K, B0, sigma0=s0, gain=1.0)
    assert L == pytest.approx(0.5 * (I - M) ** 2 / v + 0.5 * math.log(v), rel=1e-14)
    # gain and flat: v = sigma0^2/F^2 + M/(G F)
    G, F = 2.0, 1.25
    cfg = oracle.RefConfig(1, 1, 1, sigma0=s0, gain=G, flat=np.array([[F]], np.float32))
    L, g = oracle.eval_loss_grad(cfg, np.array([[Rv]], np.float32), np.array([[I]], np.float32),
                                 np.array([K, B0], np.float32))
    v = s0 ** 2 / F ** 2 + M / (G * F)
    assert L[0] == pytest.approx(0.5 * (I - M) ** 2 / v + 0.5 * math.log(v), rel=1e-14)
    # dL/dM by differentiating the closed form by hand: -(r/v) - r^2 b/(2 v^2) + b/(2v)
    r, b = I - M, 1.0 / (G * F)
    dLdM = -r / v - r * r * b / (2 * v * v) + b / (2 * v)
    assert g[0][1] == pytest.approx(dLdM, rel=1e-13)
    assert g[0][0] == pytest.approx(dLdM * Rv, rel=1e-13)


def test_constant_reference_closed_form():
    """R == const, I == const: L = N_valid [ r^2/(2v) + ln(v)/2 ] and g_K = N w R, g_B0 = N w."""
    n, m = 10, 3
    R = np.full((n, n), 50.0, np.float32)
    I = np.full((n, n), 70.0, np.float32)
    th = np.concatenate([np.full(m * m, 0.125), [1.5]]).astype(np.float32)
    M = 50.0 * 0.125 * 9 + 1.5
    v = 16.0 + M / 2.0
    N = n_valid(n, m)
    L, g = oracle.eval_loss_grad(_cfg(n, m, sigma0=4.0, gain=2.0), R, I, th)
    assert L[0] == pytest.approx(N * (0.5 * (70 - M) ** 2 / v + 0.5 * math.log(v)), rel=1e-13)
    r, b = 70 - M, 0.5
    w = -r / v - r * r * b / (2 * v * v) + b / (2 * v)
    assert np.allclose(g[0][:-1], N * w * 50.0, rtol=1e-12)
    assert g[0][-1] == pytest.approx(N * w, rel=1e-12)


def test_negative_model_reading_R1():
    """R1: the photon term uses max(M, 0) and its derivative vanishes there."""
    I, Rv, K, B0, s0 = 1.0, 10.0, -1.0, 2.0, 3.0      # M = -8
    L, g = _single_pixel(I, Rv, K, B0, sigma0=s0, gain=1.0)
    v = s0 ** 2
    assert L == pytest.approx(0.5 * 81.0 / v + 0.5 * math.log(v), rel=1e-14)
    assert g[1] == pytest.approx(-9.0 / v, rel=1e-14)


def test_fixed_mode_drops_log_term():
    """FIXED mode: L = chi^2/2 only (Eq. 5; reading R3), w = -r/v."""
    cfg = oracle.RefConfig(1, 1, 1, noise=oracle.NOISE_FIXED)
    L, g = oracle.eval_loss_grad(cfg, np.array([[10.0]], np.float32), np.array([[25.0]], np.float32),
                                 np.array([2.0, 1.0], np.float32), var=np.array([[4.0]], np.float32))
    assert L[0] == pytest.approx(0.5 * 16.0 / 4.0)
    assert g[0][1] == pytest.approx(-4.0 / 4.0)
    assert g[0][0] == pytest.approx(-10.0)


# ---------------------------------------------------------------- Huber, Eq. 12-14
def test_huber_branches_and_continuity(golden):
    """Eq. 12: quadratic for |z| <= c, c(|z| - c/2) beyond; equal values c^2/2
    and equal slopes c at |z| = c.  Catches a wrong branch constant or sign of psi."""
    c = golden["huber_c_default"]
    assert oracle.RefConfig(1, 1, 1).huber_c == c                      # API default
    cfg = oracle.RefConfig(1, 1, 1, loss=oracle.LOSS_HUBER, huber_c=c, noise=oracle.NOISE_FIXED)
    one = np.array([[1.0]], np.float32)

    def L_of(z):   # R = 1, K = 0, B0 = 0, var = 1 => z = I
        L, g = oracle.eval_loss_grad(cfg, one, np.array([[z]], np.float32),
                                     np.array([0.0, 0.0], np.float32), var=one)
        return L[0], g[0][1]

    for z in (0.3, -0.9, 1.0):
        z32 = float(np.float32(z))
        assert L_of(z)[0] == pytest.approx(0.5 * z32 * z32, rel=1e-14)
        assert L_of(z)[1] == pytest.approx(-z32, rel=1e-14)          # dL/dB0 = -psi(z)/s
    for z in (2.0, -3.5, 40.0):
        assert L_of(z)[0] == pytest.approx(c * (abs(z) - 0.5 * c), rel=1e-14)
        assert L_of(z)[1] == pytest.approx(-math.copysign(c, z), rel=1e-14)
    eps = 1e-3
    lo, hi = L_of(c - eps), L_of(c + eps)
    assert abs(hi[0] - lo[0]) < 2.1 * eps * c                          # continuous
    assert abs(hi[1] - lo[1]) < 2.1 * eps                              # C^1


def test_huber_equals_gaussian_for_large_c():
    R, I, th = _rand_problem()
    cg = _cfg(12, 3, sigma0=5.0)
    ch = _cfg(12, 3, sigma0=5.0, loss=oracle.LOSS_HUBER, huber_c=1e6)
    Lg, gg = oracle.eval_loss_grad(cg, R, I, th)
    Lh, gh = oracle.eval_loss_grad(ch, R, I, th)
    assert Lg[0] == Lh[0] and np.array_equal(gg, gh)
    # and differs (is smaller) once c bites
    ch = _cfg(12, 3, sigma0=5.0, loss=oracle.LOSS_HUBER, huber_c=0.5)
    Lh2, _ = oracle.eval_loss_grad(ch, R, I, th)
    assert Lh2[0] < Lg[0]


def test_huber_Q_constant(golden):
    """Eq. 14 is the log of the integral of exp(-rho_c); c -> inf gives
    (N/2) ln 2 pi."""
    c = golden["huber_c_default"]
    integral, _ = scipy.integrate.quad(
        lambda z: math.exp(-(0.5 * z * z if abs(z) <= c else c * (abs(z) - 0.5 * c))), -60, 60,
        points=[-c, c])
    assert oracle.huber_Q(c, 1.0) == pytest.approx(math.log(integral), rel=1e-10)
    assert oracle.huber_Q(c, 7.0) == pytest.approx(7.0 * math.log(integral), rel=1e-10)
    assert oracle.huber_Q(50.0, 10.0) == pytest.approx(5.0 * math.log(2 * math.pi), rel=1e-12)


# ---------------------------------------------------------------- Laplacian regularisation, Eq. 20-21
def _laplacian_matrix(m):
    """Eq. 21 written out: (N_K+1) x (N_K+1), L_uu = number of adjacent kernel pixels,
    L_uv = -1 for adjacent kernel pixels (4 edge neighbours, reading R14), zero row / column for B0."""
    nk = m * m
    L = np.zeros((nk + 1, nk + 1))
    for a in range(m):
        for b in range(m):
            u = a * m + b
            for da, db in ((-1, 0), (1, 0), (0, -1), (0, 1)):
                aa, bb = a + da, b + db
                if 0 <= aa < m and 0 <= bb < m:
                    L[u, u] += 1
                    L[u, aa * m + bb] = -1
    return L


def test_laplacian_penalty_matches_eq20_matrix_form():
    """Eq. 20: L = L0 + lambda N_data theta' L' L theta.  The oracle applies the stencil; the
    expected value is the explicit matrix product.  Catches a wrong neighbour count at the kernel border, a
    penalty on B0, a missing factor 2 in the gradient and a wrong N_data."""
    n, m, lam = 13, 5, 0.7
    R, I, th = _rand_problem(n, m, seed=4)
    c0 = _cfg(n, m, sigma0=5.0)
    c1 = _cfg(n, m, sigma0=5.0, lambda_reg=lam)
    L0, g0 = oracle.eval_loss_grad(c0, R, I, th)
    L1, g1 = oracle.eval_loss_grad(c1, R, I, th)
    Lm = _laplacian_matrix(m)
    assert np.array_equal(Lm, Lm.T) and np.linalg.eigvalsh(Lm).min() > -1e-12        # symmetric, PSD
    t = th.astype(np.float64)
    N = n_valid(n, m)
    pen = lam * N * t @ Lm.T @ Lm @ t
    assert L1[0] - L0[0] == pytest.approx(pen, rel=1e-10)
    assert np.allclose(g1[0] - g0[0], 2 * lam * N * (Lm.T @ Lm @ t), rtol=1e-9, atol=1e-12 * np.abs(g1).max())
    assert g1[0][-1] == g0[0][-1]                                                     # B0 is not penalised
    # a flat kernel has zero Laplacian everywhere, border included
    flat = np.concatenate([np.full(m * m, 0.125), [1.0]]).astype(np.float32)
    assert oracle.eval_loss_grad(c1, R, I, flat)[0][0] == oracle.eval_loss_grad(c0, R, I, flat)[0][0]


# ---------------------------------------------------------------- polynomial background, Eq. 18-19
def _bg_numpy(n_r, n_c, d, b):
    """Eq. 18-19 with numpy: eta = (x - x_c)/N_x, xi = (y - y_c)/N_y, x = column, y = row,
    centre = ((N-1)/2), coefficient order m = 0..d outer, n = 0..d-m inner (reading R18)."""
    y, x = np.mgrid[0:n_r, 0:n_c].astype(np.float64)
    eta = (x - (n_c - 1) / 2) / n_c
    xi = (y - (n_r - 1) / 2) / n_r
    B = np.zeros((n_r, n_c))
    t = 0
    for mm in range(d + 1):
        for nn in range(d - mm + 1):
            B += b[t] * eta ** mm * xi ** nn
            t += 1
    assert t == (d + 1) * (d + 2) // 2
    return B, eta, xi


@pytest.mark.parametrize("d", [1, 2, 3])
def test_polynomial_background_model_and_gradient(d):
    """K = delta => M = crop(R) + B(x, y); dL/db_mn = sum_V w eta^m xi^n.  Catches swapped x / y, a wrong
    centre or normalisation, a wrong coefficient order and a missing basis factor in the gradient."""
    n_r, n_c, m, h = 11, 14, 3, 1
    rng = np.random.default_rng(10 + d)
    R = (100 + 50 * rng.random((n_r, n_c))).astype(np.float32)
    I = (150 + 50 * rng.random((n_r, n_c))).astype(np.float32)
    nb = (d + 1) * (d + 2) // 2
    b = (rng.normal(0, 8, nb)).astype(np.float32)
    K = np.zeros((m, m), np.float32); K[h, h] = 1.0
    th = np.concatenate([K.ravel(), b])
    cfg = oracle.RefConfig(n_r, n_c, m, sigma0=5.0, gain=1.5, bg_degree=d)
    assert cfg.n_params == m * m + nb
    B, eta, xi = _bg_numpy(n_r, n_c, d, b.astype(np.float64))
    M = oracle.model(cfg, R, th)
    assert np.allclose(M, R[h:-h, h:-h].astype(np.float64) + B[h:-h, h:-h], rtol=1e-13, atol=1e-11)
    # gradient of the background coefficients from w, rebuilt from the model by hand (D1, Gaussian, MODEL noise)
    L, g = oracle.eval_loss_grad(cfg, R, I, th)
    v = 25.0 + M / 1.5
    r = I[h:-h, h:-h].astype(np.float64) - M
    w = -r / v + (1 / (2 * 1.5 * v)) * (1 - r * r / v)
    assert L[0] == pytest.approx((0.5 * r * r / v + 0.5 * np.log(v)).sum(), rel=1e-13)
    t = 0
    for mm in range(d + 1):
        for nn in range(d - mm + 1):
            assert g[0][m * m + t] == pytest.approx((w * eta[h:-h, h:-h] ** mm * xi[h:-h, h:-h] ** nn).sum(), rel=1e-10, abs=1e-12)
            t += 1
    # d = 0 inside the same code path is the scalar B0
    cfg0 = oracle.RefConfig(n_r, n_c, m, sigma0=5.0, gain=1.5)
    th0 = np.concatenate([K.ravel(), b[:1]])
    b1 = b.copy(); b1[1:] = 0
    assert np.array_equal(oracle.model(cfg0, R, th0), oracle.model(cfg, R, np.concatenate([K.ravel(), b1])))


# ---------------------------------------------------------------- difference image and fit-quality metrics
def test_difference_image_and_mfb_mfv():
    """D = I - M; MFB, MFV of Eq. 29-30 against numpy mean / var(ddof = 1) of
    eps = D / sigma with sigma from Eq. 6 at the model.  Catches N vs N-1, a missing mask, sigma vs sigma^2 and
    a difference image written outside the valid region."""
    n, m, h = 14, 3, 1
    R, I, th = _rand_problem(n, m, seed=9)
    rng = np.random.default_rng(2)
    flat = (0.9 + 0.2 * rng.random((n, n))).astype(np.float32)
    mask = (rng.random((n, n)) > 0.2).astype(np.uint8)
    cfg = oracle.RefConfig(n, n, m, sigma0=4.0, gain=1.7, flat=flat)
    D, met = oracle.difference_image(cfg, R, I, th, mask=mask)
    K = th[:-1].astype(np.float64).reshape(m, m)
    M = scipy.signal.correlate2d(R.astype(np.float64), K, mode="valid") + float(th[-1])
    Dn = np.zeros((n, n)); Dn[h:-h, h:-h] = I.astype(np.float64)[h:-h, h:-h] - M
    assert np.allclose(D, Dn, rtol=0, atol=1e-10) and np.all(D[0] == 0) and np.all(D[:, -1] == 0)
    F = flat.astype(np.float64)[h:-h, h:-h]
    sig = np.sqrt(16.0 / F ** 2 + M / (1.7 * F))
    use = mask[h:-h, h:-h] == 1
    eps = (Dn[h:-h, h:-h] / sig)[use]
    assert met[0] == eps.size
    assert met[1] == pytest.approx(eps.mean(), rel=1e-12)
    assert met[2] == pytest.approx(eps.var(ddof=1), rel=1e-12)
    assert met[3] == pytest.approx((eps ** 2).sum(), rel=1e-12)


# ---------------------------------------------------------------- covariance (Eq. 16-17)
def _spd(n, seed, cond=1e4):
    rng = np.random.default_rng(seed)
    Q, _ = np.linalg.qr(rng.normal(size=(n, n)))
    ev = np.exp(rng.uniform(0.0, math.log(cond), n))
    return (Q * ev) @ Q.T, ev


def test_covariance_closed_form_2x2_and_diagonal():
    """[[a, b], [b, d]]^-1 = [[d, -b], [-b, a]] / (ad - b^2) (a swapped or unsigned off-diagonal fails); a diagonal
    H gives sigma_p = 1/sqrt(H_pp) (a missing square root, or sigma taken from H instead of H^-1, fails)."""
    a, b, d = 4.0, 1.5, 3.0
    cov, sig, info = oracle.covariance(np.array([[a, b], [b, d]]), 1)
    det = a * d - b * b
    np.testing.assert_allclose(cov, np.array([[d, -b], [-b, a]]) / det, rtol=1e-14)
    np.testing.assert_allclose(sig, [math.sqrt(d / det), math.sqrt(a / det)], rtol=1e-14)
    assert info[0] == 1.0 and info[4] == 1.0
    assert info[1] == pytest.approx(math.log(det), rel=1e-14)
    assert info[2] == pytest.approx(math.sqrt(d / det), rel=1e-14)        # u = (1, 0): sigma_P = sigma_0
    np.testing.assert_allclose(info[3], 1.0 / np.linalg.eigvalsh(np.array([[a, b], [b, d]])).max(), rtol=1e-12)
    h = np.array([4.0, 0.25, 100.0, 1.0])
    cov, sig, info = oracle.covariance(np.diag(h), 3)
    np.testing.assert_allclose(sig, 1.0 / np.sqrt(h), rtol=1e-15)
    assert info[2] == pytest.approx(math.sqrt((1.0 / h[:3]).sum()), rel=1e-14)   # independent terms add in variance
    assert info[3] == pytest.approx(0.01, rel=1e-14)


@pytest.mark.parametrize("n,seed", [(5, 0), (50, 1), (123, 2)])
def test_covariance_against_numpy_spd(n, seed):
    """numpy.linalg (LAPACK) inverse, log-determinant and spectrum of a random SPD matrix with known eigenvalues."""
    H, ev = _spd(n, seed)
    nk = n - 1
    cov, sig, info = oracle.covariance(H, nk)
    ref = np.linalg.inv(H)
    scale = np.sqrt(np.outer(np.diag(ref), np.diag(ref)))
    assert (np.abs(cov - ref) / scale).max() < 1e-9
    np.testing.assert_allclose(H @ cov, np.eye(n), atol=1e-9)
    np.testing.assert_allclose(sig, np.sqrt(np.diag(ref)), rtol=1e-9)
    assert info[0] == 1.0 and info[4] == 1.0
    assert info[1] == pytest.approx(np.log(ev).sum(), rel=1e-10)          # planted spectrum, not a library call
    assert info[3] == pytest.approx(1.0 / ev.max(), rel=1e-8)
    u = np.zeros(n); u[:nk] = 1.0
    assert info[2] == pytest.approx(math.sqrt(u @ ref @ u), rel=1e-8)


def test_covariance_validity_flags():
    """a negative determinant, or any eigenvalue <= 0, makes Sigma invalid.  One negative eigenvalue
    flips the determinant; two leave it positive, so only the eigenvalue test catches that case."""
    rng = np.random.default_rng(7)
    Q, _ = np.linalg.qr(rng.normal(size=(6, 6)))
    for ev, sign in (([3, 2, 1, 0.5, 0.1, -0.2], -1.0), ([3, 2, 1, 0.5, -0.1, -0.2], 1.0)):
        ev = np.array(ev, float)
        H = (Q * ev) @ Q.T
        cov, sig, info = oracle.covariance(H, 5)
        assert info[0] == 0.0
        assert info[4] == sign
        assert info[3] == pytest.approx((1.0 / ev).min(), rel=1e-10)
        assert info[1] == pytest.approx(np.log(np.abs(ev)).sum(), rel=1e-10)
        np.testing.assert_allclose(H @ cov, np.eye(6), atol=1e-10)         # the inverse itself still exists
    cov, sig, info = oracle.covariance(np.array([[1.0, 2.0], [2.0, 4.0]]), 1)   # singular
    assert info[0] == 0.0


def test_covariance_of_planted_linear_model():
    """For a linear model y = X theta + N(0, s^2) the Fisher matrix is X'X / s^2 and the covariance of the estimate is
    s^2 (X'X)^-1 -- the textbook least-squares result; the empirical scatter of repeated fits must agree with sigma
    (a covariance taken from H instead of its inverse, or a missing square root, fails by orders of magnitude)."""
    rng = np.random.default_rng(11)
    X = rng.normal(size=(400, 4)); s = 0.3
    H = X.T @ X / s ** 2
    _, sig, info = oracle.covariance(H, 4)
    th = np.array([np.linalg.lstsq(X, X @ np.ones(4) + s * rng.normal(size=400), rcond=None)[0] for _ in range(3000)])
    np.testing.assert_allclose(th.std(axis=0), sig, rtol=0.06)
    assert th.sum(axis=1).std() == pytest.approx(info[2], rel=0.06)
