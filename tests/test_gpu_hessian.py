"""GPU-vs-oracle parity of dia_hessian (Eq. 15-17), through the C ABI.

Both sides evaluate the closed form sum_V h X X' (D3), the device in float32 per pixel with FP64
partial sums, the oracle in FP64.  Entries are compared in the metric that matters for the covariance:
  e_H = max_pq |H_gpu - H_or|_pq / sqrt(H_or,pp H_or,qq)  <= 2e-6
and the uncertainties the paper reports (sigma_P, sigma_B0, Eq. 17) must agree to 2e-5 relative.
"""
import numpy as np
import pytest

import oracle
from workloads import make_workload

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL_H = 2e-6
TOL_SIGMA = 2e-5


@pytest.fixture(scope="module")
def dia():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    import paper_2104_13715_b200 as dia
    dia.load_library()
    return dia


def _dev(a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda().contiguous()


def _e_H(Hg, Ho):
    d = np.sqrt(np.abs(np.diag(Ho)))
    return float(np.abs((Hg - Ho) / np.outer(d, d)).max())


def _sigmas(H, nk):
    """Eq. 16-17: covariance = H^-1; sigma of P = sum K (a linear combination) and of B0."""
    np.linalg.cholesky(H)                      # the positive-definiteness check of PAPER.md:183
    cov = np.linalg.inv(H)
    one = np.zeros(H.shape[0])
    one[:nk] = 1.0
    return float(np.sqrt(one @ cov @ one)), float(np.sqrt(cov[nk, nk]))


@pytest.mark.parametrize("c,n,m,E", [(0, None, None, 16), (1, 256, 15, 16), (4, 192, 19, 1), (4, 333, 11, 7),
                                     (0, 90, 5, 1), (0, 100, 3, 4), (0, 72, 1, 2)])
def test_hessian_plain_objective(dia, c, n, m, E):
    """Gaussian loss, noise model of Eq. 6, at the fitted theta (the MLE of Eq. 15); max_epochs = 1 walks the
    single-launch path, 333 the cp.async staging path and a chunk size that does not divide 2 np; m >= 5 takes the
    tensor-core kernel (m = 5: 26 of its 128 operand rows in use), m = 3 and m = 1 are handles whose evaluations run
    eval_small_kernel while the Hessian takes the block kernel and the fused kernel."""
    w = make_workload(c, n=n, m=m, n_epochs=1)
    cfg = oracle.RefConfig(w.n, w.n, w.m, sigma0=w.sigma0, gain=w.gain)
    h = dia.Handle(_dev(w.R), w.m, max_epochs=E, sigma0=w.sigma0, gain=w.gain)
    if E > 1:
        thg, _ = h.fit(_dev(w.I), _dev(w.theta0), dia.FitOpts.default())
        th = thg.cpu().numpy()[0]
    else:
        th = w.theta_true[0].astype(np.float32)
    Ho = oracle.hessian(cfg, w.R, w.I[0], th)
    Hg = h.hessian(_dev(w.I[0]), _dev(th)).cpu().numpy()
    assert np.array_equal(Hg, Hg.T)
    e = _e_H(Hg, Ho)
    nk = w.m * w.m
    sPg, sBg = _sigmas(Hg, nk)
    sPo, sBo = _sigmas(Ho, nk)
    print(f"hessian c{c} n={w.n} m={w.m}: e_H={e:.2e}  sigma_P {sPg:.6e} ({sPo:.6e})  sigma_B0 {sBg:.5e} ({sBo:.5e})")
    assert e <= TOL_H
    assert abs(sPg - sPo) <= TOL_SIGMA * sPo and abs(sBg - sBo) <= TOL_SIGMA * sBo
    Hg2 = h.hessian(_dev(w.I[0]), _dev(th)).cpu().numpy()
    assert np.array_equal(Hg, Hg2)             # deterministic
    h.close()


def test_hessian_huber_mask_flat_background_penalty(dia):
    """Every option at once: Huber loss, flat field and mask (c3), a degree-1 background and the Laplacian
    penalty, whose second derivative is 2 lambda N L'L."""
    w = make_workload(3, n=200, m=9, n_epochs=1)
    lam, d = 0.5, 1
    cfg = oracle.RefConfig(w.n, w.n, w.m, loss=oracle.LOSS_HUBER, huber_c=1.345, sigma0=w.sigma0, gain=w.gain,
                           flat=w.flat, bg_degree=d, lambda_reg=lam)
    h = dia.Handle(_dev(w.R), w.m, max_epochs=8, loss=dia.LOSS_HUBER, huber_c=1.345, sigma0=w.sigma0,
                   gain=w.gain, flat=_dev(w.flat), bg_degree=d, lambda_reg=lam)
    th = np.concatenate([w.theta_true[0], [3.0, -2.0]]).astype(np.float32)
    mask = (np.ones((w.n, w.n), np.uint8) if w.mask is None else w.mask[0]).copy()
    # The second derivative of Huber's rho jumps at |z| = c (Eq. 12): a pixel whose |z| sits within
    # float32 rounding of the threshold may take the other branch on the device, and one such pixel moves H by its
    # whole X X'/v.  The branch is a decision taken in the arithmetic's own precision, so pixels the oracle finds
    # within 1e-3 of the threshold leave the comparison (masked on both sides); what is compared is unique.
    D, _ = oracle.difference_image(cfg, w.R, w.I[0], th, mask=mask)
    M = w.I[0].astype(np.float64) - D
    F = w.flat.astype(np.float64)
    z = D / np.sqrt(w.sigma0 ** 2 / F ** 2 + np.maximum(M, 0.0) / (w.gain * F))
    near = np.abs(np.abs(z) - 1.345) < 1e-3
    print(f"hessian huber: {int((near & (mask != 0)).sum())} pixels within 1e-3 of the Huber threshold are masked out")
    mask[near] = 0
    Ho = oracle.hessian(cfg, w.R, w.I[0], th, mask=mask)
    Hg = h.hessian(_dev(w.I[0]), _dev(th), mask=_dev(mask)).cpu().numpy()
    e = _e_H(Hg, Ho)
    print(f"hessian huber+mask+flat+bg+penalty: e_H={e:.2e}")
    assert e <= TOL_H
    nk = w.m * w.m
    sPg, sBg = _sigmas(Hg, nk)
    sPo, sBo = _sigmas(Ho, nk)
    assert abs(sPg - sPo) <= TOL_SIGMA * sPo and abs(sBg - sBo) <= TOL_SIGMA * sBo
    h.close()


def test_hessian_fixed_variance_is_normal_matrix(dia):
    """DIA_NOISE_FIXED, Gaussian loss: H = X' diag(1/var) X, the B08 normal matrix, whatever theta is."""
    w = make_workload(0, n=150, m=7, n_epochs=1)
    var = (w.sigma0 ** 2 + np.clip(w.I[0], 0, None) / w.gain).astype(np.float32)
    cfg = oracle.RefConfig(w.n, w.n, w.m, noise=oracle.NOISE_FIXED)
    h = dia.Handle(_dev(w.R), w.m, max_epochs=4, noise=dia.NOISE_FIXED)
    th = w.theta_true[0].astype(np.float32)
    Ho = oracle.hessian(cfg, w.R, w.I[0], th, var=var)
    H1 = h.hessian(_dev(w.I[0]), _dev(th), var=_dev(var)).cpu().numpy()
    H2 = h.hessian(_dev(w.I[0]), _dev(w.theta0[0]), var=_dev(var)).cpu().numpy()
    print(f"hessian fixed variance: e_H {_e_H(H1, Ho):.2e}")
    assert _e_H(H1, Ho) <= TOL_H
    assert np.array_equal(H1, H2)


def test_hessian_argument_errors(dia):
    w = make_workload(0, n_epochs=2)
    R2 = np.stack([w.R, w.R])
    h = dia.Handle(_dev(R2), w.m, max_epochs=2, sigma0=w.sigma0, gain=w.gain)
    with pytest.raises(dia.DiaError):
        h.hessian(_dev(w.I[0]), _dev(w.theta_true[0].astype(np.float32)))
    h.close()


@pytest.mark.parametrize("tc", ["1", "0"])
@pytest.mark.parametrize("grid_limit", [1, 5])
def test_hessian_many_tiles_per_cta(dia, monkeypatch, grid_limit, tc):
    """Test hook DIA_GRID_LIMIT: one or five CTAs walk through all 36 tiles of a 400^2 image, so every CTA
    accumulates its FP64 partials over many tiles (the launch shape of a 4096^2 image: 4096 tiles on 147 or 296 CTAs) and
    restages its single R / I buffer between them; both paths: hess_tc_kernel (one type at m = 9) and, with
    DIA_HESS_TC=0, hess_block_kernel, whose 81 kernel-pixel rows in launches of 32 leave a ragged last one."""
    monkeypatch.setenv("DIA_GRID_LIMIT", str(grid_limit))
    monkeypatch.setenv("DIA_HESS_TC", tc)
    w = make_workload(4, n=400, m=9, n_epochs=1)
    cfg = oracle.RefConfig(w.n, w.n, w.m, sigma0=w.sigma0, gain=w.gain)
    h = dia.Handle(_dev(w.R), w.m, max_epochs=23, sigma0=w.sigma0, gain=w.gain)
    assert h.info()["grid_blocks"] == grid_limit
    th = w.theta_true[0].astype(np.float32)
    Ho = oracle.hessian(cfg, w.R, w.I[0], th)
    Hg = h.hessian(_dev(w.I[0]), _dev(th)).cpu().numpy()
    e = _e_H(Hg, Ho)
    print(f"hessian grid={grid_limit} tensor cores={tc}: e_H={e:.2e}")
    assert e <= TOL_H
    assert np.array_equal(Hg, h.hessian(_dev(w.I[0]), _dev(th)).cpu().numpy())
    h.close()


@pytest.mark.parametrize("c,n,m,outliers,sigma", [(4, 300, 19, 0, True), (1, 256, 15, 0, True), (2, 300, 13, 30, False),
                                                  (4, 200, 27, 0, False), (4, 150, 33, 0, False), (4, 112, 47, 0, False),
                                                  (0, None, None, 0, True)])
def test_hessian_tensor_core_path_against_cuda_core_path_and_oracle(dia, monkeypatch, c, n, m, outliers, sigma):
    """hess_tc_kernel (the default for m >= 5: split-float16 tcgen05 contraction, dia_hess_tc.cuh) against the FP32
    CUDA-core row passes (DIA_HESS_TC=0) and the oracle: three block types at m = 19, two at m = 13 / 15, a
    a 15-type table with single off-diagonal blocks at m = 27 (6 groups), 36 types at m = 33 (9 groups), 153 types on 153 CTAs
    at m = 47 (18 groups: more CTAs than SMs), one 128-row block at m = 7.  `outliers` plants pixels
    30 000 counts BELOW the model, whose h = d^2 l / dM^2 is negative (D3): their tile rows take the second, negated
    pass of the kernel.  The uncertainties of Eq. 17 are asserted where the Hessian tests assert them (`sigma`); the
    729-parameter kernel on a 200^2 image (cond(H) = 2e10, 42 pixels per parameter: the float32 Hessian of EITHER path is
    at the edge of positive definiteness) is compared entry by entry only."""
    w = make_workload(c, n=n, m=m, n_epochs=1)
    I = w.I[0].copy()
    if outliers:
        rng = np.random.default_rng(3)
        hh = (w.m - 1) // 2
        ys, xs = rng.integers(hh, w.n - hh, outliers), rng.integers(hh, w.n - hh, outliers)
        I[ys, xs] -= 30000.0
    huber = w.loss == "huber" and not outliers          # the planted pixels test the quadratic loss's negative h
    cfg = oracle.RefConfig(w.n, w.n, w.m, sigma0=w.sigma0, gain=w.gain, loss=oracle.LOSS_HUBER if huber else oracle.LOSS_GAUSSIAN)
    th = w.theta_true[0].astype(np.float32)
    Ho = oracle.hessian(cfg, w.R, I, th)
    H = {}
    for tc in ("1", "0"):
        monkeypatch.setenv("DIA_HESS_TC", tc)
        h = dia.Handle(_dev(w.R), w.m, max_epochs=4, sigma0=w.sigma0, gain=w.gain, loss=dia.LOSS_HUBER if huber else dia.LOSS_GAUSSIAN)
        H[tc] = h.hessian(_dev(I), _dev(th)).cpu().numpy()
        assert np.array_equal(H[tc], h.hessian(_dev(I), _dev(th)).cpu().numpy())
        h.close()
    e_tc, e_cc, e_x = _e_H(H["1"], Ho), _e_H(H["0"], Ho), _e_H(H["1"], H["0"])
    nk = w.m * w.m
    print(f"hessian c{c} n={w.n} m={w.m} outliers={outliers}: e_H tensor cores {e_tc:.2e}, CUDA cores {e_cc:.2e}, one against the "
          f"other {e_x:.2e}; negative-h pixels matter: {bool(outliers)}")
    assert not np.array_equal(H["1"], H["0"])          # the hook really switches the path
    assert e_tc <= TOL_H and e_cc <= TOL_H and e_x <= TOL_H
    if sigma:
        sPo, sBo = _sigmas(Ho, nk)
        for tc in ("1", "0"):
            sPg, sBg = _sigmas(H[tc], nk)
            print(f"   tensor cores={tc}: sigma_P {sPg:.6e} ({sPo:.6e}: {abs(sPg / sPo - 1):.1e})  sigma_B0 {sBg:.5e} ({sBo:.5e}: "
                  f"{abs(sBg / sBo - 1):.1e})  cond(H) {np.linalg.cond(Ho):.1e}")
            assert abs(sPg - sPo) <= TOL_SIGMA * sPo and abs(sBg - sBo) <= TOL_SIGMA * sBo
