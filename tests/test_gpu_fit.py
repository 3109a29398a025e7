"""GPU-vs-oracle parity of dia_fit (on-device Adam -> L-BFGS), through the C ABI.

Fit parity protocol: same theta_init and options on both sides.
  strict     |dP| <= 1e-4 |P|,  |dB0| <= 1e-4 max(|B0|, 1),  max|dK| <= 1e-4 max|K_or|
             required (a) in lock-step mode (force_*_iters: both sides take exactly the same steps, which
             pins the device Adam / L-BFGS arithmetic) and (b) for free-running fits driven to convergence.
  stopped    |dL| <= 1e-3 |L|,  |dP| <= 1e-3 |P|,  ||M_gpu - M_or||_2 <= 1e-2 ||M_or||_2
             for free-running fits under the paper's stop rule (relative loss change 1e-8).
             Fixed-step L-BFGS is not monotone and the rule fires on the first chance |dL| < 1e-8 |L|, usually
             while the flat directions of K are still undetermined at the 1e-2 level (cond(H) 1e6..1e13); the
             iteration at which it fires depends on every rounding, on either side.  The stopped K, B0 and the
             iteration counts are therefore reported, not asserted ("parity unpinned");
             what is asserted is that both sides stop legitimately at statistically equivalent models.
"""
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


OPT_KEYS = ("lr_kernel", "lr_b0", "adam_beta1", "adam_beta2", "adam_eps", "tol_switch", "lbfgs_lr",
            "lbfgs_history", "lbfgs_backtrack", "tol_change_rel", "tol_grad_abs", "tol_grad_rel",
            "max_adam_iters", "max_lbfgs_iters", "force_adam_iters", "force_lbfgs_iters")


def _both_opts(dia, **kw):
    og, oo = dia.FitOpts.default(**kw), oracle.RefFitOpts.default(**kw)
    for k in OPT_KEYS:                       # the two libraries state the same defaults independently
        assert float(getattr(og, k)) == pytest.approx(float(getattr(oo, k)), rel=1e-7), k
    return og, oo


def _fit_both(dia, w, og, oo, var=None, noise_fixed=False):
    lossg = dia.LOSS_HUBER if w.loss == "huber" else dia.LOSS_GAUSSIAN
    losso = oracle.LOSS_HUBER if w.loss == "huber" else oracle.LOSS_GAUSSIAN
    cfg = oracle.RefConfig(w.n, w.n, w.m, loss=losso, sigma0=w.sigma0, gain=w.gain, flat=w.flat,
                           noise=oracle.NOISE_FIXED if noise_fixed else oracle.NOISE_MODEL)
    h = dia.Handle(_dev(w.R), w.m, max_epochs=w.n_epochs, loss=lossg, sigma0=w.sigma0, gain=w.gain,
                   flat=_dev(w.flat), noise=dia.NOISE_FIXED if noise_fixed else dia.NOISE_MODEL)
    tho, ro = oracle.fit(cfg, w.R, w.I, w.theta0, oo, mask=w.mask, var=var)
    thg, rg = h.fit(_dev(w.I), _dev(w.theta0), og, mask=_dev(w.mask), var=_dev(var))
    h.close()
    return tho, ro, thg.cpu().numpy(), rg


def _diffs(tho, ro, thg, rg, e):
    Ko, Kg = tho[e][:-1].astype(np.float64), thg[e][:-1].astype(np.float64)
    dK = np.abs(Kg - Ko).max() / np.abs(Ko).max()
    dP = abs(rg[e].photometric_scale - ro[e].photometric_scale) / abs(ro[e].photometric_scale)
    dB = abs(float(thg[e][-1]) - float(tho[e][-1])) / max(abs(float(tho[e][-1])), 1.0)
    dL = abs(rg[e].loss - ro[e].loss) / abs(ro[e].loss) if ro[e].loss != 0 else abs(rg[e].loss)
    return dK, dP, dB, dL


def _report(tag, e, d, ro, rg):
    print(f"{tag} e{e}: dK={d[0]:.2e} dP={d[1]:.2e} dB0={d[2]:.2e} dL={d[3]:.2e} "
          f"gpu(adam={rg[e].n_adam}, lbfgs={rg[e].n_lbfgs}, evals={rg[e].n_evals}, st={rg[e].status}) "
          f"oracle(adam={ro[e].n_adam}, lbfgs={ro[e].n_lbfgs}, evals={ro[e].n_evals}, st={ro[e].status})")


def _assert_fit_close(tho, ro, thg, rg, tag, tol=1e-4):
    """strict criterion"""
    for e in range(tho.shape[0]):
        d = _diffs(tho, ro, thg, rg, e)
        _report(tag, e, d, ro, rg)
        assert d[1] <= tol and d[2] <= tol and d[0] <= tol, f"{tag} epoch {e}"
        assert rg[e].photometric_scale == pytest.approx(thg[e][:-1].astype(np.float64).sum(), rel=1e-6)  # Eq. 3


def _assert_fit_model_close(w, tho, ro, thg, rg, tag):
    """stopped criterion: both fits stop legitimately at statistically equivalent models"""
    cfg = oracle.RefConfig(w.n, w.n, w.m)
    for e in range(tho.shape[0]):
        d = _diffs(tho, ro, thg, rg, e)
        _report(tag, e, d, ro, rg)
        Mo, Mg = oracle.model(cfg, w.R, tho[e]), oracle.model(cfg, w.R, thg[e])
        dM = np.linalg.norm(Mg - Mo) / np.linalg.norm(Mo)
        print(f"{tag} e{e}: ||dM||/||M|| = {dM:.2e}")
        assert d[3] <= 1e-3 and d[1] <= 1e-3 and dM <= 1e-2, f"{tag} epoch {e}"
        assert rg[e].status in (0, 1) and ro[e].status in (0, 1)


@pytest.mark.parametrize("n_adam,n_lbfgs,backtrack", [(1, 0, 0), (5, 0, 0), (40, 0, 0), (0, 3, 0), (0, 3, 1),
                                                       (30, 12, 0), (30, 12, 1)])
def test_fit_lockstep(dia, n_adam, n_lbfgs, backtrack):
    """Fixed iteration counts: both sides take exactly the same steps, so the iterates differ only by
    the FP32 evaluation error of the gradient.  Catches any mistake in the device Adam / two-loop
    recursion / step-size / history bookkeeping."""
    w = make_workload(0)
    og, oo = _both_opts(dia, force_adam_iters=n_adam, force_lbfgs_iters=n_lbfgs, lbfgs_backtrack=backtrack)
    tho, ro, thg, rg = _fit_both(dia, w, og, oo)
    assert rg[0].n_adam == ro[0].n_adam == n_adam
    assert rg[0].n_lbfgs == ro[0].n_lbfgs
    assert rg[0].n_evals == ro[0].n_evals
    _assert_fit_close(tho, ro, thg, rg, f"lockstep {n_adam}/{n_lbfgs}/bt{backtrack}")


def test_fit_free_running_config0_paper_stop_rule(dia):
    """BASELINE config 0 (128^2, m = 7, Gaussian likelihood, seed 0), paper settings."""
    w = make_workload(0)
    og, oo = _both_opts(dia)
    tho, ro, thg, rg = _fit_both(dia, w, og, oo)
    _assert_fit_model_close(w, tho, ro, thg, rg, "c0 free")
    # and lands on the planted parameters within the noise (P = 1.2)
    assert rg[0].photometric_scale == pytest.approx(1.2, abs=0.02)


def test_fit_free_running_config0_converged(dia):
    """Same fit driven to convergence (loss-change rule tightened to 1e-13): the objective is convex
    (PAPER.md:135), so both optimisers must reach the same minimiser -- strict criterion."""
    w = make_workload(0)
    og, oo = _both_opts(dia, tol_change_rel=1e-13, max_lbfgs_iters=3000)
    tho, ro, thg, rg = _fit_both(dia, w, og, oo)
    _assert_fit_close(tho, ro, thg, rg, "c0 converged")


def test_fit_planted_recovery_fixed_mode(dia):
    """Noise-free target, FIXED variance (reading R12): the minimum is theta_true with L = 0
    (paper tests (i)-(iii), report eps_P ~ 4e-7 at FP32)."""
    w = make_workload(0, noise=False)
    var = np.full(w.I.shape, 25.0, np.float32)
    og, oo = _both_opts(dia, lr_b0=1.0)
    tho, ro, thg, rg = _fit_both(dia, w, og, oo, var=var, noise_fixed=True)
    P_true = w.theta_true[0][:-1].sum()
    print(f"planted: gpu eps_P={abs(rg[0].photometric_scale - P_true) / P_true:.2e} "
          f"oracle eps_P={abs(ro[0].photometric_scale - P_true) / P_true:.2e} "
          f"gpu max|dK|={np.abs(thg[0][:-1] - w.theta_true[0][:-1]).max():.2e}")
    assert abs(rg[0].photometric_scale - P_true) / P_true < 1e-4
    assert abs(ro[0].photometric_scale - P_true) / P_true < 1e-4
    assert np.abs(thg[0][:-1] - w.theta_true[0][:-1]).max() < 1e-3 * w.theta_true[0][:-1].max()


def test_fit_batched_epochs_match_oracle_and_singles(dia):
    """Batched fit (subsystem 3): epochs converge after different iteration counts inside one graph
    launch; each must equal, bit for bit, the fit of that epoch alone."""
    w = make_workload(4, n=160, n_epochs=3, m=9)
    og, oo = _both_opts(dia, max_adam_iters=3000)
    tho, ro, thg, rg = _fit_both(dia, w, og, oo)
    _assert_fit_model_close(w, tho, ro, thg, rg, "c4-small batched")
    h = dia.Handle(_dev(w.R), w.m, max_epochs=1, sigma0=w.sigma0, gain=w.gain)
    for e in range(3):
        th1, r1 = h.fit(_dev(w.I[e:e + 1]), _dev(w.theta0[e:e + 1]), og)
        assert np.array_equal(th1.cpu().numpy()[0], thg[e])
        assert (r1[0].n_adam, r1[0].n_lbfgs, r1[0].n_evals) == (rg[e].n_adam, rg[e].n_lbfgs, rg[e].n_evals)
    h.close()


def test_fit_many_small_pairs(dia):
    """One reference per epoch: 6 independent 142^2 / 19x19 stamps (the paper's stamp shape)
    fitted in one graph launch, lock-step against the oracle stamp by stamp.  8 Adam steps: strict criterion.
    (Longer horizons are not asserted at m = 19: Adam normalises every component of the gradient, so the
    components that are cancelling sums -- accurate to 1e-7 of their scale S_p but only to ~1e-4 of their own
    value -- get steps that differ at that level, and the difference accumulates: measured dK = 1.7e-4 after
    20 steps, 1.3e-2 after 200.)  With 20 Adam + 3 L-BFGS steps the batch must still stop at equivalent models."""
    from test_gpu_parity import _stamp_batch
    S, n, m = 6, 142, 19
    R, I, th0, tht = _stamp_batch(S, n, m)
    cfg = oracle.RefConfig(n, n, m, sigma0=5.0, gain=1.0)
    h = dia.Handle(_dev(R), m, max_epochs=S, sigma0=5.0, gain=1.0)
    for n_lbfgs in (0, 3):
        og, oo = _both_opts(dia, force_adam_iters=8 if n_lbfgs == 0 else 20, force_lbfgs_iters=n_lbfgs)
        thg, rg = h.fit(_dev(I), _dev(th0), og)
        thg = thg.cpu().numpy()
        for k in range(S):
            tho, ro = oracle.fit(cfg, R[k], I[k], th0[k], oo)
            assert rg[k].n_evals == ro[0].n_evals
            if n_lbfgs == 0:
                _assert_fit_close(tho, ro, thg[k:k + 1], rg[k:k + 1], f"stamp {k}")
            else:
                d = _diffs(tho, ro, thg[k:k + 1], rg[k:k + 1], 0)
                _report(f"stamp {k} +lbfgs", 0, d, ro, rg[k:k + 1])
                assert d[3] <= 5e-2 and d[1] <= 5e-2      # reported; far from the optimum fixed-step L-BFGS amplifies
    h.close()


def test_fit_with_laplacian_regularisation(dia):
    """Eq. 20 inside dia_fit: lock-step against the oracle (strict), then free-running under the paper's
    stop rule.  The penalty lifts the flat directions of K; it does not touch the scale-background valley (a constant
    kernel offset against B0: L 1 = 0), so the free-running part uses the background-subtracted reference of the
    paper's practice, where B0 is well determined too -- then the stopped iterate itself meets the strict
    criterion (with the sky left in the reference dB0 hovers around 1e-4: tests/test_gpu_fit_protocol.py)."""
    lam = 10.0
    w = make_workload(0)
    cfg = oracle.RefConfig(w.n, w.n, w.m, sigma0=w.sigma0, gain=w.gain, lambda_reg=lam)
    h = dia.Handle(_dev(w.R), w.m, sigma0=w.sigma0, gain=w.gain, lambda_reg=lam)
    og, oo = _both_opts(dia, force_adam_iters=30, force_lbfgs_iters=10)
    tho, ro = oracle.fit(cfg, w.R, w.I, w.theta0, oo)
    thg, rg = h.fit(_dev(w.I), _dev(w.theta0), og)
    _assert_fit_close(tho, ro, thg.cpu().numpy(), rg, "lambda lockstep")
    h.close()
    w = make_workload(0, sky_subtract=True)
    h = dia.Handle(_dev(w.R), w.m, sigma0=w.sigma0, gain=w.gain, lambda_reg=lam)
    og, oo = _both_opts(dia)
    tho, ro = oracle.fit(cfg, w.R, w.I, w.theta0, oo)
    thg, rg = h.fit(_dev(w.I), _dev(w.theta0), og)
    thg = thg.cpu().numpy()
    d = _diffs(tho, ro, thg, rg, 0)
    _report("lambda free", 0, d, ro, rg)
    assert d[3] <= 1e-5 and d[0] <= 1e-4 and d[1] <= 1e-4 and d[2] <= 1e-4      # strict, free-running
    # the penalised loss is larger than the plain one at the same theta, and the fitted kernel is smoother
    cfg0 = oracle.RefConfig(w.n, w.n, w.m, sigma0=w.sigma0, gain=w.gain)
    L_pen, _ = oracle.eval_loss_grad(cfg, w.R, w.I, thg[0])
    L_0, _ = oracle.eval_loss_grad(cfg0, w.R, w.I, thg[0])
    assert L_pen[0] > L_0[0] and rg[0].loss == pytest.approx(L_pen[0], rel=1e-6)
    h.close()


def test_fit_polynomial_background(dia):
    """Eq. 18-19 inside dia_fit: a planted background gradient is absorbed by the degree-1 coefficients.
    Lock-step against the oracle (strict), then a free-running regularised fit recovers the planted slope."""
    w = make_workload(0)
    n, m = w.n, w.m
    y, x = np.mgrid[0:n, 0:n].astype(np.float64)
    eta, xi = (x - (n - 1) / 2) / n, (y - (n - 1) / 2) / n
    I = (w.I[0].astype(np.float64) + 30.0 * eta - 18.0 * xi).astype(np.float32)[None]     # b_10 = 30, b_01 = -18
    th0 = np.concatenate([w.theta0[0], [0.0, 0.0]]).astype(np.float32)[None]               # [K, b_00, b_01, b_10]
    lam = 10.0
    cfg = oracle.RefConfig(n, n, m, sigma0=w.sigma0, gain=w.gain, bg_degree=1, lambda_reg=lam)
    h = dia.Handle(_dev(w.R), m, sigma0=w.sigma0, gain=w.gain, bg_degree=1, lambda_reg=lam)
    og, oo = _both_opts(dia, force_adam_iters=30, force_lbfgs_iters=6)
    tho, ro = oracle.fit(cfg, w.R, I, th0, oo)
    thg, rg = h.fit(_dev(I), _dev(th0), og)
    thg = thg.cpu().numpy()
    assert rg[0].n_evals == ro[0].n_evals
    assert np.abs(thg[0][:m * m] - tho[0][:m * m]).max() <= 1e-4 * np.abs(tho[0][:m * m]).max()
    assert np.abs(thg[0][m * m:] - tho[0][m * m:]).max() <= 1e-4 * max(1.0, np.abs(tho[0][m * m:]).max())
    assert rg[0].photometric_scale == pytest.approx(ro[0].photometric_scale, rel=1e-4)
    og, oo = _both_opts(dia, lr_b0=10.0)
    tho, ro = oracle.fit(cfg, w.R, I, th0, oo)
    thg, rg = h.fit(_dev(I), _dev(th0), og)
    thg = thg.cpu().numpy()
    print("bg fit gpu b =", thg[0][m * m:], "oracle b =", tho[0][m * m:], "P", rg[0].photometric_scale, ro[0].photometric_scale,
          "iters", rg[0].n_evals, ro[0].n_evals)
    assert rg[0].status in (0, 1)
    assert abs(thg[0][m * m + 2] - 30.0) < 3.0 and abs(thg[0][m * m + 1] + 18.0) < 3.0      # b_10, b_01 within noise
    assert rg[0].photometric_scale == pytest.approx(ro[0].photometric_scale, rel=1e-3)
    h.close()


def test_fit_constant_bank_graph_matches_shared_memory_graph(dia, monkeypatch):
    """dia_fit on a large image refreshes the constant block inside the graph before every evaluation (pack
    kernel + device-to-device copy to the symbol) and drops finished epochs from it; the result must equal the
    shared-memory variant bit for bit, epochs finishing at different iterations included."""
    w = make_workload(4, n=600, n_epochs=3, m=9)           # 10 x 10 tiles
    og = dia.FitOpts.default(max_adam_iters=400, max_lbfgs_iters=40)
    h = dia.Handle(_dev(w.R), w.m, max_epochs=3, sigma0=w.sigma0, gain=w.gain)
    thc, rc = h.fit(_dev(w.I), _dev(w.theta0), og)
    h.close()
    monkeypatch.setenv("DIA_DISABLE_CONST", "1")
    h2 = dia.Handle(_dev(w.R), w.m, max_epochs=3, sigma0=w.sigma0, gain=w.gain)
    ths, rs = h2.fit(_dev(w.I), _dev(w.theta0), og)
    h2.close()
    assert torch.equal(thc, ths)
    for a, b in zip(rc, rs):
        assert (a.n_adam, a.n_lbfgs, a.n_evals, a.status, a.loss) == (b.n_adam, b.n_lbfgs, b.n_evals, b.status, b.loss)
    assert len({r.n_evals for r in rc}) > 1                 # the epochs did stop at different iterations


def test_fit_host_chunked_pipeline_matches_device_fit(dia):
    """dia_fit_host (C ABI; Handle.fit_host marshals) cuts the batch into groups whose host->device copies overlap the
    fit of the previous group; the fitted parameters must equal those of one device-resident dia_fit over the whole
    batch.  dia_eval_loss_grad_host likewise against dia_eval_loss_grad, with pageable host memory too."""
    w = make_workload(4, n=200, n_epochs=9, m=7)
    og = dia.FitOpts.default(force_adam_iters=40, force_lbfgs_iters=10)
    h = dia.Handle(_dev(w.R), w.m, max_epochs=9, sigma0=w.sigma0, gain=w.gain)
    thd, rd = h.fit(_dev(w.I), _dev(w.theta0), og)
    hI, hth = torch.from_numpy(w.I).pin_memory(), torch.from_numpy(w.theta0).pin_memory()
    for chunks in (None, 1, 3, 9):
        thh, rh, h2d, d2h = h.fit_host(hI, hth, og, chunks=chunks)
        assert torch.equal(thh, thd.cpu())
        assert [r.n_evals for r in rh] == [r.n_evals for r in rd] and [r.loss for r in rh] == [r.loss for r in rd]
        assert h2d == w.I.nbytes + w.theta0.nbytes
    Ld, gd = h.eval_loss_grad(_dev(w.I), _dev(w.theta0))
    for hI2, hth2 in ((hI, hth), (torch.from_numpy(w.I.copy()), torch.from_numpy(w.theta0.copy()))):     # pinned, pageable
        Lh, gh, _, d2h = h.eval_loss_grad_host(hI2, hth2)
        assert torch.equal(Lh, Ld.cpu()) and torch.equal(gh, gd.cpu()) and d2h == 8 * (9 + 9 * 50)
    Lh, gh, _, _ = h.eval_loss_grad_host(hI[:2], hth[:2])                            # fewer epochs than max_epochs
    assert torch.equal(Lh, Ld.cpu()[:2]) and torch.equal(gh, gd.cpu()[:2])
    mask = (np.random.default_rng(1).random(w.I.shape) > 0.01).astype(np.uint8)
    thm, rm = h.fit(_dev(w.I), _dev(w.theta0), og, mask=_dev(mask))
    thh, rh, h2d, _ = h.fit_host(hI, hth, og, mask_host=torch.from_numpy(mask).pin_memory())
    assert torch.equal(thh, thm.cpu()) and h2d == w.I.nbytes + w.theta0.nbytes + mask.nbytes
    h.close()


def test_fit_huber_with_cosmic_rays(dia):
    """BASELINE config 2 shape at reduced size: robust objective, 0.1 % cosmic-ray hits, no mask."""
    w = make_workload(2, n=200, m=9)
    og, oo = _both_opts(dia, max_adam_iters=4000)
    tho, ro, thg, rg = _fit_both(dia, w, og, oo)
    _assert_fit_model_close(w, tho, ro, thg, rg, "c2-small huber")
    assert rg[0].photometric_scale == pytest.approx(1.1, abs=0.03)


def test_fit_mask_and_flat(dia):
    """BASELINE config 3 shape at reduced size: per-pixel flat field and 2 % masked pixels."""
    w = make_workload(3, n=200, m=9)
    og, oo = _both_opts(dia, max_adam_iters=4000)
    tho, ro, thg, rg = _fit_both(dia, w, og, oo)
    _assert_fit_model_close(w, tho, ro, thg, rg, "c3-small")


def test_fit_is_deterministic_and_reusable(dia):
    """Two fits through the same handle (the cached graph is relaunched) give identical bits."""
    w = make_workload(0, n=96, m=5)
    h = dia.Handle(_dev(w.R), w.m, sigma0=w.sigma0, gain=w.gain)
    og = dia.FitOpts.default()
    I, th0 = _dev(w.I), _dev(w.theta0)
    th1, r1 = h.fit(I, th0, og)
    th2, r2 = h.fit(I, th0, og)
    assert torch.equal(th1, th2) and r1[0].loss == r2[0].loss and r1[0].n_evals == r2[0].n_evals
    h.close()


def test_fit_nonfinite_status(dia):
    """sigma0 = 0 and a negative model make ln v non-finite (reading R1): status NONFINITE, no hang."""
    w = make_workload(0, n=64, m=5)
    h = dia.Handle(_dev(w.R), 5, sigma0=0.0, gain=1.0)
    th0 = w.theta0.copy()
    th0[:, :-1] = -0.04
    th, r = h.fit(_dev(w.I), _dev(th0), dia.FitOpts.default())
    assert r[0].status == 3 and r[0].n_evals == 1
    h.close()


@pytest.mark.parametrize("m,lam", [(35, 0.0), (47, 0.0), (47, 0.05)])
def test_fit_lockstep_large_kernels(dia, m, lam):
    """Kernels of the paper's real-data fits (median 27 x 27, maximum 47 x 47 on 142^2 stamps):
    m >= 33 runs one CTA per SM, and more than 1024 parameters take the wide instantiation of the optimiser
    kernel.  Two stamps, lock-step Adam + L-BFGS, with and without the Laplacian penalty."""
    w = make_workload(0, n=142, m=m, n_epochs=2)
    og, oo = _both_opts(dia, force_adam_iters=8, force_lbfgs_iters=4)
    cfg = oracle.RefConfig(w.n, w.n, w.m, sigma0=w.sigma0, gain=w.gain, lambda_reg=lam)
    h = dia.Handle(_dev(w.R), w.m, max_epochs=2, sigma0=w.sigma0, gain=w.gain, lambda_reg=lam)
    assert h.info()["grid_blocks"] <= 148          # one resident CTA per SM
    tho, ro = oracle.fit(cfg, w.R, w.I, w.theta0, oo)
    thg, rg = h.fit(_dev(w.I), _dev(w.theta0), og)
    h.close()
    assert [r.n_evals for r in rg] == [r.n_evals for r in ro]
    _assert_fit_close(tho, ro, thg.cpu().numpy(), rg, f"lockstep m={m} lambda={lam}")


@pytest.mark.parametrize("c,n,m,E", [(0, None, None, 1), (0, 100, 5, 3), (4, 142, 19, 5), (1, 190, 9, 2), (2, 120, 9, 2)])
def test_fit_cluster_kernel_matches_graph_loop(dia, monkeypatch, c, n, m, E):
    """Small image pairs with the plain objective are fitted inside one kernel, one thread-block cluster per epoch
    (csrc/dia_fit_cluster.cuh: tiles resident in shared memory, cluster barriers instead of launches).  Same device
    functions, same orders: for image pairs whose tiles sit on different CTAs in the graph loop the fitted parameters,
    iteration counts and losses must be bit-identical to it (test hook DIA_DISABLE_CLUSTER=1), free-running and in
    lock-step; (190^2: 3 x 3 = 9 tiles exceed the portable cluster size and take the graph loop on both sides).
    The graph loop it is compared with is the one over the generic kernel, whose device functions the cluster kernel
    shares: DIA_DISABLE_SMALL=1 keeps the m = 5 case off eval_small_kernel (other arithmetic order, equal to rounding:
    tests/test_gpu_small_kernels.py)."""
    w = make_workload(c, n=n, m=m, n_epochs=E)
    monkeypatch.setenv("DIA_DISABLE_SMALL", "1")
    outs = []
    for disable in ("0", "1"):
        monkeypatch.setenv("DIA_DISABLE_CLUSTER", disable)
        h = dia.Handle(_dev(w.R), w.m, max_epochs=E, sigma0=w.sigma0, gain=w.gain,
                       loss=dia.LOSS_HUBER if w.loss == "huber" else dia.LOSS_GAUSSIAN)      # (config 2: the robust objective)
        res = []
        for og in (dia.FitOpts.default(max_adam_iters=2500, max_lbfgs_iters=60),
                   dia.FitOpts.default(force_adam_iters=25, force_lbfgs_iters=7, lbfgs_backtrack=1)):
            th, r = h.fit(_dev(w.I), _dev(w.theta0), og)
            res.append((th.cpu().numpy(), [(x.n_adam, x.n_lbfgs, x.n_evals, x.status, x.loss, x.grad_inf_norm,
                                            x.photometric_scale) for x in r]))
        h.close()
        outs.append(res)
    for (tha, ra), (thb, rb) in zip(*outs):
        assert ra == rb
        assert np.array_equal(tha, thb)
    assert outs[0][0][1][0][2] > 30          # the free-running fit did iterate
