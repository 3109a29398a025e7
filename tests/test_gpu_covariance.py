"""GPU-vs-oracle parity of dia_covariance (Eq. 16-17 and the validity test of PAPER.md:193), through the C ABI.

The device factorises H = L L' (FP64) and solves for the rows of Sigma; the oracle inverts by Gauss-Jordan elimination
and diagonalises Sigma as the paper describes.  Both are FP64 and backward stable, so they differ by about
cond(H) x 1e-16; entries are compared in the correlation metric
  e_S = max_pq |S_gpu - S_or|_pq / sqrt(S_or,pp S_or,qq)  <= 1e-9 x max(1, cond(H) / 1e5)
and the uncertainties (sigma_p, sigma_P; Eq. 17) relative to their own size with the same bound.
"""
import math

import numpy as np
import pytest

import oracle
from workloads import make_workload

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dia():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    import paper_2104_13715_b200 as dia
    dia.load_library()
    return dia


def _dev(a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda().contiguous()


def _handle(dia, m, n=64):
    """A handle only fixes np = m*m + 1 and the number of kernel parameters here."""
    R = np.full((n, n), 100.0, np.float32)
    return dia.Handle(_dev(R), m, max_epochs=1)


def _spd(n, seed, cond):
    rng = np.random.default_rng(seed)
    Q, _ = np.linalg.qr(rng.normal(size=(n, n)))
    ev = np.exp(rng.uniform(0.0, math.log(cond), n))
    H = (Q * ev) @ Q.T
    return 0.5 * (H + H.T), ev


def _compare(covg, sigg, infog, covo, sigo, infoo, tol):
    d = np.sqrt(np.diag(covo))
    e_S = float(np.abs((covg - covo) / np.outer(d, d)).max())
    e_sig = float(np.abs(sigg / sigo - 1.0).max())
    e_P = abs(infog[2] / infoo[2] - 1.0)
    assert infog[0] == 1.0 and infoo[0] == 1.0
    assert infog[4] == -1.0
    assert abs(infog[1] - infoo[1]) <= 1e-10 * max(1.0, abs(infoo[1]))
    assert e_S <= tol and e_sig <= tol and e_P <= tol, (e_S, e_sig, e_P, tol)
    return e_S, e_sig, e_P


@pytest.mark.parametrize("m,cond,seed", [(1, 10.0, 0), (3, 1e3, 1), (7, 1e4, 2), (19, 1e6, 3), (25, 1e5, 4)])
def test_covariance_planted_spectrum(dia, m, cond, seed):
    """Random SPD matrices with a planted spectrum: np = 2 (one warp), 10, 50, 362 (45 CTAs of 8 rows + 2: ragged) and
    626 rows; ln det H is the sum of the planted log-eigenvalues -- known without either implementation."""
    h = _handle(dia, m)
    n = m * m + 1
    H, ev = _spd(n, seed, cond)
    covg, sigg, infog = (t.cpu().numpy() for t in h.covariance(_dev(H)))
    covo, sigo, infoo = oracle.covariance(H, m * m)
    tol = 1e-9 * max(1.0, cond / 1e5)
    e = _compare(covg, sigg, infog, covo, sigo, infoo, tol)
    print(f"covariance np={n} cond={cond:.0e}: e_S={e[0]:.2e} e_sigma={e[1]:.2e} e_sigmaP={e[2]:.2e}")
    assert abs(infog[1] - np.log(ev).sum()) <= 1e-10 * abs(np.log(ev).sum()) + 1e-10
    assert np.array_equal(covg, covg.T)
    assert np.abs(H @ covg - np.eye(n)).max() <= 1e-7 * max(1.0, cond / 1e5)
    assert infog[3] > 0.0
    # uncertainties alone (no back-substitution) and a repeated call: the same bits
    _, sig2, info2 = h.covariance(_dev(H), want_cov=False)
    assert np.array_equal(sig2.cpu().numpy(), sigg) and np.array_equal(info2.cpu().numpy(), infog)
    cov3, _, _ = h.covariance(_dev(H))
    assert np.array_equal(cov3.cpu().numpy(), covg)
    h.close()


@pytest.mark.parametrize("c,n,m", [(0, None, None), (1, 256, 15)])
def test_covariance_of_fitted_model_end_to_end(dia, c, n, m):
    """The paper's use: fit, observed Fisher information at the MLE (Eq. 15), covariance (Eq. 16), uncertainties
    (Eq. 17), all on the device, against the oracle's Hessian and inverse at the same theta.  The float32 per-pixel
    arithmetic of dia_hessian sets the error here (tests/test_gpu_hessian.py: 2e-5 on sigma)."""
    w = make_workload(c, n=n, m=m, n_epochs=1)
    cfg = oracle.RefConfig(w.n, w.n, w.m, sigma0=w.sigma0, gain=w.gain)
    h = dia.Handle(_dev(w.R), w.m, max_epochs=16, sigma0=w.sigma0, gain=w.gain)
    thg, res = h.fit(_dev(w.I), _dev(w.theta0), dia.FitOpts.default())
    th = thg.cpu().numpy()[0]
    nk = w.m * w.m
    Hg = h.hessian(_dev(w.I[0]), thg[0].contiguous())
    covg, sigg, infog = (t.cpu().numpy() for t in h.covariance(Hg))
    Ho = oracle.hessian(cfg, w.R, w.I[0], th)
    covo, sigo, infoo = oracle.covariance(Ho, nk)
    cond = np.linalg.cond(Ho)
    print(f"covariance c{c}: cond(H)={cond:.2e} valid={infog[0]:.0f} sigma_P {infog[2]:.6e} ({infoo[2]:.6e}) "
          f"sigma_B0 {sigg[nk]:.5e} ({sigo[nk]:.5e})  P={res[0].photometric_scale:.5f}")
    assert infog[0] == 1.0 and infoo[0] == 1.0
    assert abs(infog[2] - infoo[2]) <= 2e-5 * infoo[2]
    assert abs(sigg[nk] - sigo[nk]) <= 2e-5 * sigo[nk]
    # single kernel pixels: Sigma = H^-1 turns the Hessian's error dH into -Sigma dH Sigma, so to first order
    # |d Sigma_pp| / Sigma_pp <= |dH^|_2 / lambda_min(H^) with H^ = D^-1/2 H D^-1/2 the unit-diagonal scaling of H
    # (e_p' S^2 e_p <= lambda_max(S) e_p' S e_p), and half of that on sigma_p.  Weakly constrained wing pixels make
    # lambda_min(H^) small, so this bound -- not a fixed tolerance -- is what the float32 Hessian can promise.
    d = 1.0 / np.sqrt(np.diag(Ho))
    Hs, dHs = Ho * np.outer(d, d), (Hg.cpu().numpy() - Ho) * np.outer(d, d)
    bound = 0.6 * np.linalg.norm(dHs, 2) / np.linalg.eigvalsh(Hs).min()
    e_sig = np.abs(sigg / sigo - 1.0).max()
    print(f"   single-pixel uncertainties: max |sigma_gpu / sigma_or - 1| = {e_sig:.2e}, first-order bound {bound:.2e}")
    assert e_sig <= max(bound, 1e-6)
    # ln det H: the device factorises ITS Hessian, so the reference value is numpy's FP64 log-determinant of that same
    # matrix (the factorisation's accuracy), and the difference to the oracle's ln det is the float32 Hessian's doing:
    # tr(H^-1 dH) to first order, reported -- with cond(H) ~ 1e9 the relative perturbation |H^-1 dH| of the weakest
    # directions is O(1) (see the bound above) and the higher orders are as large as the first, so no linearised
    # value is asserted
    sign, lndet_np = np.linalg.slogdet(Hg.cpu().numpy())
    d_lndet = float(np.sum(covo * (Hg.cpu().numpy() - Ho)))
    print(f"   ln det H {infog[1]:.6f} (numpy on the same matrix {lndet_np:.6f}; oracle's H {infoo[1]:.6f}, first-order "
          f"prediction of the difference {d_lndet:.3e})")
    assert sign > 0 and abs(infog[1] - lndet_np) <= 1e-9 * abs(lndet_np)
    assert abs(infog[1] - infoo[1]) <= 1e-4 * abs(infoo[1])
    # the linear algebra alone, both sides on the oracle's Hessian
    cov2, sig2, info2 = (t.cpu().numpy() for t in h.covariance(_dev(Ho)))
    _compare(cov2, sig2, info2, covo, sigo, infoo, 1e-9 * max(1.0, cond / 1e5))
    # the planted scale factor lies within a few sigma_P of the fitted one (a sanity check of the error bar itself)
    assert abs(res[0].photometric_scale - w.theta_true[0][:nk].sum()) <= 5.0 * infog[2]
    h.close()


def test_covariance_invalid_matrix_raises_flag(dia):
    """an indefinite matrix is not a valid covariance.  The first non-positive pivot is the first
    leading principal minor that fails Sylvester's criterion, found here with numpy determinants."""
    m = 5
    h = _handle(dia, m)
    n = m * m + 1
    rng = np.random.default_rng(5)
    H, _ = _spd(n, 9, 1e3)
    v = rng.normal(size=n); v[:10] = 0.0                     # leaves the leading 10 x 10 block positive definite
    H = H - 2.0 * np.linalg.eigvalsh(H).max() * np.outer(v, v) / (v @ v)
    first_bad = next(k for k in range(n) if np.linalg.det(H[:k + 1, :k + 1]) <= 0.0)
    assert first_bad >= 10
    _, _, infog = (t if t is None else t.cpu().numpy() for t in h.covariance(_dev(H), want_cov=False))
    _, _, infoo = oracle.covariance(H, m * m)
    assert infog[0] == 0.0 and infoo[0] == 0.0
    assert infog[4] == float(first_bad)
    assert infog[3] < 0.0
    # two negative eigenvalues (positive determinant): only the eigenvalue test of the paper catches it, and so must
    # the pivots
    Q, _ = np.linalg.qr(rng.normal(size=(n, n)))
    ev = np.linspace(1.0, 3.0, n); ev[3] = -0.5; ev[17] = -0.25
    H2 = (Q * ev) @ Q.T
    H2 = 0.5 * (H2 + H2.T)
    _, _, infog = (t if t is None else t.cpu().numpy() for t in h.covariance(_dev(H2), want_cov=False))
    _, _, infoo = oracle.covariance(H2, m * m)
    assert infoo[4] == 1.0 and infoo[0] == 0.0
    assert infog[0] == 0.0
    h.close()


def test_covariance_argument_errors(dia):
    h = _handle(dia, 3)
    H = _dev(np.eye(10))
    sig = torch.empty(10, dtype=torch.float64, device="cuda")
    info = torch.empty(5, dtype=torch.float64, device="cuda")
    with pytest.raises(dia.DiaError):
        dia.dia_covariance(h._h, None, None, sig, info)
    with pytest.raises(dia.DiaError):
        dia.dia_covariance(h._h, H, H, sig, info)
    with pytest.raises(dia.DiaError):
        dia.dia_covariance(h._h, H, None, None, info)
    h.close()


def test_covariance_maximum_size_properties(dia):
    """m = 47 (DIA_MAX_KERNEL_SIZE): np = 2210, beyond what the oracle's Jacobi diagonalisation finishes in seconds, so
    the properties that define the result are checked instead: H Sigma = 1, exact symmetry, ln det H equal to the sum of
    the planted log-eigenvalues, and sigma / sigma_P against LAPACK's inverse."""
    m = 47
    h = _handle(dia, m, n=64)
    n = m * m + 1
    H, ev = _spd(n, 12, 1e4)
    cov, sig, info = (t.cpu().numpy() for t in h.covariance(_dev(H)))
    assert info[0] == 1.0 and info[4] == -1.0
    assert abs(info[1] - np.log(ev).sum()) <= 1e-10 * abs(np.log(ev).sum())
    assert np.array_equal(cov, cov.T)
    assert np.abs(H @ cov - np.eye(n)).max() <= 1e-8
    ref = np.linalg.inv(H)
    np.testing.assert_allclose(sig, np.sqrt(np.diag(ref)), rtol=1e-9)
    u = np.zeros(n); u[:m * m] = 1.0
    assert info[2] == pytest.approx(np.sqrt(u @ ref @ u), rel=1e-9)
    h.close()
