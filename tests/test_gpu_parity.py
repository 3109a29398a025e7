"""GPU-vs-oracle parity of dia_eval_loss_grad, through the C ABI (python -m pytest -m gpu).

Protocol: on the same seeded inputs
  loss      |L_gpu - L_or| <= 1e-5 |L_or|                                   at every point
  gradient  e_norm = max|dg| / max|g_or| <= 1e-5                            where the gradient is far from
                                                                            cancelling (theta_init)
            e_S    = max_p |dg_p| / S_p <= 1e-5, S_p = sum_V |w| |X_p|      at near-stationary points
                                                                            (theta_true and perturbations),
                                                                            e_norm reported
and repeated evaluations are bit-identical.
"""
import numpy as np
import pytest

import oracle
from workloads import make_workload

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL = 1e-5


@pytest.fixture(scope="module")
def dia():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    import paper_2104_13715_b200 as dia
    dia.load_library()
    return dia


def _dev(a, dtype=None):
    if a is None:
        return None
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda().contiguous()


def _ref_cfg(w, **kw):
    loss = oracle.LOSS_HUBER if w.loss == "huber" else oracle.LOSS_GAUSSIAN
    args = dict(loss=loss, sigma0=w.sigma0, gain=w.gain, flat=w.flat)
    args.update(kw)
    return oracle.RefConfig(w.n, w.n, w.m, **args)


def _handle(dia, w, max_epochs=None, **kw):
    args = dict(max_epochs=max_epochs or w.n_epochs,
                loss=dia.LOSS_HUBER if w.loss == "huber" else dia.LOSS_GAUSSIAN,
                sigma0=w.sigma0, gain=w.gain, flat=_dev(w.flat))
    args.update(kw)
    return dia.Handle(_dev(w.R), w.m, **args)


def _points(w):
    """P0 = theta_init, P1 = theta_true, P2 = theta_true (1 + 1e-3 xi)."""
    rng = np.random.default_rng(77 + w.config.index)
    p2 = w.theta_true * (1.0 + 1e-3 * rng.standard_normal(w.theta_true.shape))
    return [("P0", w.theta0.astype(np.float32), "norm"),
            ("P1", w.theta_true.astype(np.float32), "S"),
            ("P2", p2.astype(np.float32), "S")]


def _compare(Lg, gg, Lo, go, So, kind, tag):
    Lg, gg = Lg.cpu().numpy(), gg.cpu().numpy()
    for e in range(Lo.shape[0]):
        assert abs(Lg[e] - Lo[e]) <= TOL * abs(Lo[e]), f"{tag} epoch {e}: loss {Lg[e]} vs {Lo[e]}"
        d = np.abs(gg[e] - go[e])
        e_norm = d.max() / np.abs(go[e]).max()
        e_S = (d / So[e]).max()
        print(f"{tag} e{e}: dL/L={abs(Lg[e]-Lo[e])/abs(Lo[e]):.2e} e_norm={e_norm:.2e} e_S={e_S:.2e}")
        assert e_S <= TOL, f"{tag} epoch {e}: e_S = {e_S:.3e}"
        if kind == "norm":
            assert e_norm <= TOL, f"{tag} epoch {e}: e_norm = {e_norm:.3e}"


CASES = [  # (config, n, n_epochs): element-by-element sizes the oracle finishes in seconds;
    (0, None, None),     # several 64x64 tiles plus a ragged tail in every case
    (1, None, None),
    (2, 600, None),
    (3, 500, None),
    (4, 333, 3),         # odd n: unaligned rows (scalar cp.async path)
    (4, 520, 2),
]


@pytest.mark.parametrize("c,n,E", CASES)
def test_eval_parity(dia, c, n, E):
    w = make_workload(c, n=n, n_epochs=E)
    h = _handle(dia, w)
    cfg = _ref_cfg(w)
    I, mask = _dev(w.I), _dev(w.mask)
    for name, th, kind in _points(w):
        Lo, go, So = oracle.eval_loss_grad(cfg, w.R, w.I, th, mask=w.mask, want_scale=True)
        Lg, gg = h.eval_loss_grad(I, _dev(th), mask=mask)
        Lg2, gg2 = h.eval_loss_grad(I, _dev(th), mask=mask)
        torch.cuda.synchronize()
        assert torch.equal(Lg, Lg2) and torch.equal(gg, gg2), "evaluation is not deterministic"
        _compare(Lg, gg, Lo, go, So, kind, f"c{c} n={w.n} {name}")
    h.close()


@pytest.mark.parametrize("c,n,m", [(0, None, None), (1, 160, 9), (2, 200, 9), (3, 160, 7)])
def test_eval_parity_at_oracle_iterates(dia, c, n, m):
    """Points P3 and P4 of the protocol: the oracle's Adam iterate at 25 % of its Adam phase
    (gradient far from cancelling: e_norm required) and the oracle's fitted theta (near-stationary: e_S
    required, e_norm reported).  The iterates come from the oracle alone."""
    w = make_workload(c, n=n, m=m, n_epochs=1)
    cfg = _ref_cfg(w)
    th4, res = oracle.fit(cfg, w.R, w.I, w.theta0, mask=w.mask)
    k = max(1, res[0].n_adam // 4)
    th3, _ = oracle.fit(cfg, w.R, w.I, w.theta0,
                        oracle.RefFitOpts.default(force_adam_iters=k, force_lbfgs_iters=0), mask=w.mask)
    h = _handle(dia, w)
    for name, th, kind in (("P3", th3, "norm"), ("P4", th4, "S")):
        th = np.asarray(th, np.float32)
        Lo, go, So = oracle.eval_loss_grad(cfg, w.R, w.I, th, mask=w.mask, want_scale=True)
        Lg, gg = h.eval_loss_grad(_dev(w.I), _dev(th), mask=_dev(w.mask))
        _compare(Lg, gg, Lo, go, So, kind, f"c{c} n={w.n} {name} (oracle Adam iterate {k} / fitted theta)")
    h.close()


@pytest.mark.parametrize("loss", ["gaussian", "huber"])
@pytest.mark.parametrize("m", [1, 3, 5, 9, 11, 13, 17, 21, 23, 27, 29, 31, 33, 35, 37, 39, 41, 43, 45, 47])
def test_eval_parity_all_kernel_sizes(dia, loss, m):
    """Every instantiated kernel size, both objectives, FIXED and MODEL noise."""
    w = make_workload(2 if loss == "huber" else 1, n=150, m=m)
    for noise in ("model", "fixed"):
        var = None
        kw = {}
        if noise == "fixed":
            var = (w.sigma0 ** 2 + np.maximum(w.I, 0.0) / w.gain).astype(np.float32)
            kw = dict(noise=dia.NOISE_FIXED)
        h = _handle(dia, w, **kw)
        cfg = _ref_cfg(w, **({"noise": oracle.NOISE_FIXED} if noise == "fixed" else {}))
        for name, th, kind in _points(w)[:2]:
            Lo, go, So = oracle.eval_loss_grad(cfg, w.R, w.I, th, var=var, want_scale=True)
            Lg, gg = h.eval_loss_grad(_dev(w.I), _dev(th), var=_dev(var))
            _compare(Lg, gg, Lo, go, So, kind, f"m={m} {loss} {noise} {name}")
        h.close()


@pytest.mark.parametrize("grid_limit,disable_tma", [(1, "0"), (3, "0"), (1, "1"), (296, "1")])
def test_many_tiles_per_cta_and_staging_paths(dia, monkeypatch, grid_limit, disable_tma):
    """Test hooks DIA_GRID_LIMIT / DIA_DISABLE_TMA: a grid of 1 or 3 CTAs makes every CTA walk through many
    tiles (double-buffer wrap-around, mbarrier phase flips, the periodic FP64 flush every 32 tiles), and the
    cp.async staging path is forced on an image whose rows are 16-byte aligned.  Results must still match the
    oracle, and the two staging paths must agree bit for bit."""
    monkeypatch.setenv("DIA_GRID_LIMIT", str(grid_limit))
    monkeypatch.setenv("DIA_DISABLE_TMA", disable_tma)
    w = make_workload(4, n=600, n_epochs=2, m=19)          # 10 x 10 tiles per epoch
    h = _handle(dia, w)
    assert h.info()["grid_blocks"] == min(grid_limit, 2 * 100)     # 2 epochs x 100 tiles of work items
    cfg = _ref_cfg(w)
    th = w.theta_true.astype(np.float32)
    Lo, go, So = oracle.eval_loss_grad(cfg, w.R, w.I, th, want_scale=True)
    Lg, gg = h.eval_loss_grad(_dev(w.I), _dev(th))
    _compare(Lg, gg, Lo, go, So, "S", f"grid={grid_limit} tma_off={disable_tma}")
    h.close()
    monkeypatch.setenv("DIA_DISABLE_TMA", "1" if disable_tma == "0" else "0")
    h2 = _handle(dia, w)
    L2, g2 = h2.eval_loss_grad(_dev(w.I), _dev(th))
    assert torch.equal(Lg, L2) and torch.equal(gg, g2)
    h2.close()


def _stamp_batch(n_stamps, n=142, m=19):
    """Independent small image pairs in the shape of the paper's stamp workloads (142^2, 19x19 kernel,
    PAPER.md:363-365): every stamp has its own reference (a different crop of a config-2 field) and target."""
    big = make_workload(2, n=512, m=m)
    from workloads import make_target, theta_init, CONFIGS
    Rs, Is, th0, tht = [], [], [], []
    for k in range(n_stamps):
        y, x = 37 * (k % 9), 41 * (k // 9 % 9)
        R = np.ascontiguousarray(big.R[y:y + n, x:x + n])
        I, th, _, _ = make_target(CONFIGS[0], 100 + k, R, m)       # Gaussian kernel, no outliers, own seed
        Rs.append(R); Is.append(I); tht.append(th.astype(np.float32)); th0.append(theta_init(R, I, m))
    return np.stack(Rs), np.stack(Is), np.stack(th0), np.stack(tht)


def test_many_small_pairs_one_reference_each(dia):
    """Batched mode with one reference per epoch (dia_config.n_refs == max_epochs): 12 independent 142^2
    stamps evaluated in one launch; every stamp must match the oracle run on that stamp alone, and the
    batch must equal the stamps evaluated one at a time, bit for bit."""
    S, n, m = 12, 142, 19
    R, I, th0, tht = _stamp_batch(S, n, m)
    h = dia.Handle(_dev(R), m, max_epochs=S, sigma0=5.0, gain=1.0)
    cfg = oracle.RefConfig(n, n, m, sigma0=5.0, gain=1.0)
    for th, kind in ((th0, "norm"), (tht, "S")):
        Lg, gg = h.eval_loss_grad(_dev(I), _dev(th))
        Lo = np.empty(S); go = np.empty((S, m * m + 1)); So = np.empty((S, m * m + 1))
        for k in range(S):
            l, g_, s_ = oracle.eval_loss_grad(cfg, R[k], I[k], th[k], want_scale=True)
            Lo[k], go[k], So[k] = l[0], g_[0], s_[0]
        _compare(Lg, gg, Lo, go, So, kind, "stamps")
    h1 = dia.Handle(_dev(R[5]), m, max_epochs=1, sigma0=5.0, gain=1.0)
    L1, g1 = h1.eval_loss_grad(_dev(I[5:6]), _dev(tht[5:6]))
    assert torch.equal(L1[0], Lg[5]) and torch.equal(g1[0], gg[5])
    h1.close()
    h.close()


@pytest.mark.parametrize("S,grid_limit", [(16, 8), (20, 8), (9, 3)])
def test_many_small_pairs_whole_epochs_per_cta(dia, monkeypatch, S, grid_limit):
    """With at least one image pair per resident CTA each CTA takes whole pairs (one change of epoch per pair, one
    column of partials) when that balances as well as dealing tiles out one by one: 16 pairs on 8 CTAs and 9 on
    3 do, 20 on 8 do not.  The test hook DIA_GRID_LIMIT stands in for a batch of several hundred pairs.
    Loss, gradient and a lock-step fit must match the oracle in both orders, and the difference image too."""
    monkeypatch.setenv("DIA_GRID_LIMIT", str(grid_limit))
    n, m = 100, 9                                          # 92^2 valid pixels: 2 x 2 tiles per pair
    R, I, th0, tht = _stamp_batch(S, n, m)
    h = dia.Handle(_dev(R), m, max_epochs=S, sigma0=5.0, gain=1.0)
    assert h.info()["grid_blocks"] == grid_limit
    cfg = oracle.RefConfig(n, n, m, sigma0=5.0, gain=1.0)
    for th, kind in ((th0, "norm"), (tht, "S")):
        Lg, gg = h.eval_loss_grad(_dev(I), _dev(th))
        Lo = np.empty(S); go = np.empty((S, m * m + 1)); So = np.empty((S, m * m + 1))
        for k in range(S):
            l, g_, s_ = oracle.eval_loss_grad(cfg, R[k], I[k], th[k], want_scale=True)
            Lo[k], go[k], So[k] = l[0], g_[0], s_[0]
        _compare(Lg, gg, Lo, go, So, kind, f"stamps S={S} grid={grid_limit}")
    opts = dia.FitOpts.default(force_adam_iters=6, force_lbfgs_iters=3)
    thg, res = h.fit(_dev(I), _dev(th0), opts)
    thg = thg.cpu().numpy()
    D, met = h.difference_image(_dev(I), _dev(tht))
    for k in (0, S // 2, S - 1):
        tho, _ = oracle.fit(cfg, R[k], I[k], th0[k], oracle.RefFitOpts.default(force_adam_iters=6, force_lbfgs_iters=3))
        assert np.abs(thg[k] - tho[0]).max() <= 1e-5 * np.abs(tho[0]).max()
        Do, mo = oracle.difference_image(cfg, R[k], I[k], tht[k])
        assert np.abs(D[k].cpu().numpy() - Do).max() <= 1e-5 * np.abs(I[k]).max()
        assert met[k].cpu().numpy() == pytest.approx(mo, rel=1e-5, abs=1e-5)
    h.close()


@pytest.mark.parametrize("c,n,m,lam", [(0, None, None, 1.0), (4, 300, 19, 0.1), (2, 200, 9, 100.0)])
def test_laplacian_regularisation_eq20(dia, c, n, m, lam):
    """Eq. 20-21: L0 + lambda N_data theta' L' L theta, evaluated on the device."""
    w = make_workload(c, n=n, m=m, n_epochs=2 if c == 4 else None)
    h = _handle(dia, w, lambda_reg=lam)
    cfg = _ref_cfg(w, lambda_reg=lam)
    cfg0 = _ref_cfg(w)
    for name, th, kind in _points(w)[:2]:
        Lo, go, So = oracle.eval_loss_grad(cfg, w.R, w.I, th, mask=w.mask, want_scale=True)
        L0, _ = oracle.eval_loss_grad(cfg0, w.R, w.I, th, mask=w.mask)
        assert np.all(Lo > L0) if name == "P1" else np.all(Lo >= L0)   # flat theta_init has zero Laplacian
        Lg, gg = h.eval_loss_grad(_dev(w.I), _dev(th), mask=_dev(w.mask))
        _compare(Lg, gg, Lo, go, So, kind, f"lambda={lam} c{c} {name}")
    h.close()


@pytest.mark.parametrize("d,c,n,m", [(1, 0, None, None), (2, 4, 333, 19), (3, 1, 300, 15), (3, 3, 260, 9)])
def test_polynomial_background_eq18(dia, d, c, n, m):
    """Eq. 18-19: spatially varying background of degree d replaces B0; the gradient gets
    (d+1)(d+2)/2 background components.  Odd n exercises the cp.async staging path, c3 the flat + mask path."""
    w = make_workload(c, n=n, m=m, n_epochs=2 if c == 4 else None)
    nb = (d + 1) * (d + 2) // 2
    rng = np.random.default_rng(40 + d)
    E = w.n_epochs
    def with_bg(th):
        b = np.concatenate([th[:, -1:], rng.normal(0, 5.0, (E, nb - 1))], axis=1)
        return np.concatenate([th[:, :-1], b], axis=1).astype(np.float32)
    h = _handle(dia, w, bg_degree=d)
    cfg = _ref_cfg(w, bg_degree=d)
    for name, th, kind in _points(w)[:2]:
        th = with_bg(np.asarray(th, np.float64))
        Lo, go, So = oracle.eval_loss_grad(cfg, w.R, w.I, th, mask=w.mask, want_scale=True)
        Lg, gg = h.eval_loss_grad(_dev(w.I), _dev(th), mask=_dev(w.mask))
        assert gg.shape[1] == w.m * w.m + nb
        _compare(Lg, gg, Lo, go, So, kind, f"bg d={d} c{c} {name}")
    h.close()


@pytest.mark.parametrize("c,n,m,d", [(0, None, None, 0), (3, 300, 11, 0), (4, 333, 19, 2), (1, 400, 15, 0)])
def test_difference_image_and_metrics(dia, c, n, m, d):
    """dia_difference_image: D = I - M element by element (float32 model against the FP64 oracle) and the
    fit-quality metrics MFB / MFV / chi^2 (Eq. 29-30), with flat + mask (c3), a polynomial
    background and the cp.async path (c4 at odd n), and after a real fit (c0)."""
    w = make_workload(c, n=n, m=m, n_epochs=2 if c == 4 else None)
    nb = (d + 1) * (d + 2) // 2
    h = _handle(dia, w, bg_degree=d)
    cfg = _ref_cfg(w, bg_degree=d)
    th = w.theta_true.astype(np.float32)
    if d > 0:
        rng = np.random.default_rng(1)
        th = np.concatenate([th, rng.normal(0, 4.0, (w.n_epochs, nb - 1)).astype(np.float32)], axis=1)
    if c == 0:                                   # difference image at the fitted parameters
        thg, _ = h.fit(_dev(w.I), _dev(w.theta0), dia.FitOpts.default())
        th = thg.cpu().numpy()
    D, met = h.difference_image(_dev(w.I), _dev(th), mask=_dev(w.mask))
    D, met = D.cpu().numpy(), met.cpu().numpy()
    hh = (w.m - 1) // 2
    for e in range(w.n_epochs):
        Do, mo = oracle.difference_image(cfg, w.R, w.I[e], th[e], mask=None if w.mask is None else w.mask[e])
        Mo = w.I[e].astype(np.float64) - Do
        # |D_gpu - D_or| against the size of the model image: float32 accumulation of M (~ 1e-6 relative)
        err = np.abs(D[e] - Do)[hh:-hh, hh:-hh] / np.maximum(np.abs(Mo[hh:-hh, hh:-hh]), 1.0)
        print(f"diff c{c} e{e}: max |dD|/|M| = {err.max():.2e}; N={met[e][0]:.0f} MFB={met[e][1]:.5f} ({mo[1]:.5f}) "
              f"MFV={met[e][2]:.5f} ({mo[2]:.5f})")
        assert err.max() <= 1e-5
        assert np.all(D[e][:hh] == 0) and np.all(D[e][:, -hh:] == 0)          # outside the valid region
        assert met[e][0] == mo[0]
        assert abs(met[e][1] - mo[1]) <= 1e-5 * max(1.0, abs(mo[1]))
        assert met[e][2] == pytest.approx(mo[2], rel=1e-5) and met[e][3] == pytest.approx(mo[3], rel=1e-5)
    if c == 0:      # a converged fit of simulated data: MFB ~ 0, MFV ~ 1 - (m^2+1)/N (Table 2)
        N = (w.n - w.m + 1) ** 2
        assert abs(met[0][1]) < 4 / np.sqrt(N) and abs(met[0][2] - (1 - 50 / N)) < 4 * np.sqrt(2 / N)
    h.close()


def test_emccd_noise_model_eq7(dia):
    """EMCCD noise model, Eq. 7: sigma^2 = E M / (G_total F) with E = 2, G_total = 25.8/300
    e-/ADU -- the affine form of Eq. 6 with no read-noise term, i.e. sigma0 = 0 and gain = G_total / E."""
    E_excess, G_total = 2.0, 25.8 / 300.0
    w = make_workload(1, n=200, m=9)
    rng = np.random.default_rng(3)
    flat = rng.uniform(0.95, 1.05, w.R.shape).astype(np.float32)
    gain = G_total / E_excess
    cfg = oracle.RefConfig(w.n, w.n, w.m, sigma0=0.0, gain=gain, flat=flat)
    th = w.theta_true.astype(np.float32)
    Lo, go, So = oracle.eval_loss_grad(cfg, w.R, w.I, th, want_scale=True)
    # the oracle's value is Eq. 7 written out: check one pixel by hand
    M = oracle.model(oracle.RefConfig(w.n, w.n, w.m), w.R, th[0])
    i, j, hh = 57, 91, 4
    v = E_excess * M[i - hh, j - hh] / (G_total * float(flat[i, j]))
    mask = np.zeros(w.I.shape, np.uint8); mask[0, i, j] = 1
    L1, _ = oracle.eval_loss_grad(cfg, w.R, w.I, th, mask=mask)
    r = float(w.I[0, i, j]) - M[i - hh, j - hh]
    assert L1[0] == pytest.approx(0.5 * r * r / v + 0.5 * np.log(v), rel=1e-9)
    for disable in ("0", "1"):
        h = dia.Handle(_dev(w.R), w.m, sigma0=0.0, gain=gain, flat=_dev(flat))
        Lg, gg = h.eval_loss_grad(_dev(w.I), _dev(th))
        _compare(Lg, gg, Lo, go, So, "S", "emccd")
        h.close()


def test_constant_bank_variant_matches_shared_memory_variant(dia, monkeypatch):
    """Long launches evaluate with the kernel pixels in the constant bank (uniform-register operands); the
    shared-memory variant (test hook DIA_DISABLE_CONST, or a handle on another stream than the one that claimed
    the block) must give the same bits, and both must match the oracle.  Handles on one stream share the block:
    interleaved evaluations of two of them with different theta must not see each other's kernel pixels."""
    w = make_workload(4, n=640, n_epochs=3, m=19)          # 3 x 100 tiles on 296 resident CTAs: two waves
    th = w.theta_true.astype(np.float32)
    cfg = _ref_cfg(w)
    Lo, go, So = oracle.eval_loss_grad(cfg, w.R, w.I, th, want_scale=True)
    h = _handle(dia, w)                                    # claims the block of m = 19 for this stream
    assert h.info()["launches_per_eval"] == 3              # pack, eval, reduce
    Lc, gc = h.eval_loss_grad(_dev(w.I), _dev(th))
    _compare(Lc, gc, Lo, go, So, "S", "const bank")
    h2 = _handle(dia, w)                                   # same stream: shares the block
    assert h2.info()["launches_per_eval"] == 3
    th_b = _dev(w.theta0)
    Lb, gb = h2.eval_loss_grad(_dev(w.I), th_b)
    for _ in range(3):                                     # interleaved, back to back on the stream
        L1, g1 = h.eval_loss_grad(_dev(w.I), _dev(th))
        L2, g2 = h2.eval_loss_grad(_dev(w.I), th_b)
        assert torch.equal(Lc, L1) and torch.equal(gc, g1)
        assert torch.equal(Lb, L2) and torch.equal(gb, g2)
    side = torch.cuda.Stream()
    h4 = _handle(dia, w, stream=side)                      # another stream: shared-memory variant
    assert h4.info()["launches_per_eval"] == 2
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        L4, g4 = h4.eval_loss_grad(_dev(w.I), _dev(th))
    side.synchronize()
    assert torch.equal(Lc, L4) and torch.equal(gc, g4)
    h.close(); h2.close(); h4.close()
    monkeypatch.setenv("DIA_DISABLE_CONST", "1")
    h3 = _handle(dia, w)
    assert h3.info()["launches_per_eval"] == 2
    L3, g3 = h3.eval_loss_grad(_dev(w.I), _dev(th))
    assert torch.equal(Lc, L3) and torch.equal(gc, g3)
    h3.close()


def test_constant_bank_two_host_threads_two_handles(dia):
    """Threading contract of include/dia.h: different handles may be driven from different host threads, also when they
    share a stream and therefore the constant block of their kernel size.  Each evaluation is three enqueues (pack,
    copy to the bank, launch); the library makes the triple atomic, so no evaluation may run with the other handle's
    kernel pixels.  Two threads, 40 evaluations each at different theta, every result bit-identical to the one
    computed alone."""
    import threading
    w = make_workload(4, n=640, n_epochs=3, m=19)
    I = _dev(w.I)
    ths = [_dev(w.theta_true.astype(np.float32)), _dev(w.theta0)]
    hs = [_handle(dia, w), _handle(dia, w)]
    assert all(h.info()["launches_per_eval"] == 3 for h in hs)
    want = [h.eval_loss_grad(I, th) for h, th in zip(hs, ths)]
    torch.cuda.synchronize()
    assert not torch.equal(want[0][0], want[1][0])
    bad, errs = [0, 0], []
    go_flag = threading.Barrier(2)

    def work(k):
        try:
            torch.cuda.set_device(0)
            go_flag.wait()
            outs = [hs[k].eval_loss_grad(I, ths[k]) for _ in range(40)]
            torch.cuda.synchronize()
            bad[k] = sum(1 for L, g in outs if not (torch.equal(L, want[k][0]) and torch.equal(g, want[k][1])))
        except Exception as exc:      # noqa: BLE001 -- reported below
            errs.append(exc)

    ts = [threading.Thread(target=work, args=(k,)) for k in range(2)]
    [t.start() for t in ts]
    [t.join() for t in ts]
    assert not errs, errs
    assert bad == [0, 0], f"evaluations that saw the other handle's kernel: {bad}"
    [h.close() for h in hs]


def test_constant_bank_variant_on_a_batch_of_medium_images(dia, monkeypatch):
    """The constant-bank variant is chosen by launch length, not image size: 24 epochs of 300^2 (25 tiles each,
    three waves of the 296 resident CTAs) use it; same bits as the shared-memory variant, and the oracle's values."""
    w = make_workload(4, n=300, n_epochs=24, m=19)
    th = w.theta_true.astype(np.float32)
    h = _handle(dia, w)
    assert h.info()["launches_per_eval"] == 3
    Lc, gc = h.eval_loss_grad(_dev(w.I), _dev(th))
    Lo, go, So = oracle.eval_loss_grad(_ref_cfg(w), w.R, w.I, th, want_scale=True)
    _compare(Lc, gc, Lo, go, So, "S", "const bank, 24 x 300^2")
    h.close()
    monkeypatch.setenv("DIA_DISABLE_CONST", "1")
    h3 = _handle(dia, w)
    assert h3.info()["launches_per_eval"] == 2
    L3, g3 = h3.eval_loss_grad(_dev(w.I), _dev(th))
    assert torch.equal(Lc, L3) and torch.equal(gc, g3)
    h3.close()


def test_rectangular_image(dia):
    w = make_workload(1, n=200, m=9)
    R, I = w.R[:137, :], w.I[:, :137, :]
    cfg = oracle.RefConfig(137, 200, 9, sigma0=w.sigma0, gain=w.gain)
    h = dia.Handle(_dev(R), 9, sigma0=w.sigma0, gain=w.gain)
    for th, kind in ((w.theta0, "norm"), (w.theta_true.astype(np.float32), "S")):
        Lo, go, So = oracle.eval_loss_grad(cfg, R, I, th, want_scale=True)
        Lg, gg = h.eval_loss_grad(_dev(I), _dev(th))
        _compare(Lg, gg, Lo, go, So, kind, "rect")
    h.close()


def test_border_poison_and_mask(dia):
    """Pixels of I / mask / var outside the valid set are never read (include/dia.h); a masked
    pixel contributes nothing (reading R4)."""
    w = make_workload(0, n=100, m=7)
    hh = 3
    h = _handle(dia, w)
    th = _dev(w.theta_true.astype(np.float32))
    L0, g0 = h.eval_loss_grad(_dev(w.I), th)
    Ip = w.I.copy()
    Ip[:, :hh, :] = np.nan; Ip[:, -hh:, :] = np.nan; Ip[:, :, :hh] = np.nan; Ip[:, :, -hh:] = np.nan
    L1, g1 = h.eval_loss_grad(_dev(Ip), th)
    assert torch.equal(L0, L1) and torch.equal(g0, g1)
    # NaN under a masked pixel must not leak
    rng = np.random.default_rng(5)
    mask = (rng.random(w.I.shape) > 0.3).astype(np.uint8)
    Ip = w.I.copy()
    Ip[mask == 0] = np.nan
    Lg, gg = h.eval_loss_grad(_dev(Ip), th, mask=_dev(mask))
    Lo, go, So = oracle.eval_loss_grad(_ref_cfg(w), w.R, w.I, w.theta_true.astype(np.float32), mask=mask,
                                       want_scale=True)
    _compare(Lg, gg, Lo, go, So, "S", "mask")
    # everything masked: exact zeros
    Lz, gz = h.eval_loss_grad(_dev(w.I), th, mask=_dev(np.zeros_like(mask)))
    assert float(Lz[0]) == 0.0 and float(gz.abs().max()) == 0.0
    h.close()


def test_minimum_size_image(dia):
    """Degenerate case n == m: a single valid pixel."""
    rng = np.random.default_rng(2)
    m = 5
    R = (100 + 50 * rng.random((m, m))).astype(np.float32)
    I = (120 + 50 * rng.random((1, m, m))).astype(np.float32)
    th = np.concatenate([np.full(m * m, 0.04), [2.0]]).astype(np.float32)
    cfg = oracle.RefConfig(m, m, m, sigma0=3.0, gain=1.5)
    Lo, go, So = oracle.eval_loss_grad(cfg, R, I, th, want_scale=True)
    h = dia.Handle(_dev(R), m, sigma0=3.0, gain=1.5)
    Lg, gg = h.eval_loss_grad(_dev(I), _dev(th))
    _compare(Lg, gg, Lo, go, So, "norm", "n==m")
    h.close()


def test_batched_equals_singles(dia):
    """Batched mode (north_star subsystem 3): one launch over E epochs == E single-epoch calls, bit for bit."""
    w = make_workload(4, n=300, n_epochs=4, m=19)
    h = _handle(dia, w)
    th = _dev(w.theta0)
    I = _dev(w.I)
    L, g = h.eval_loss_grad(I, th)
    for e in range(4):
        Le, ge = h.eval_loss_grad(I[e:e + 1].contiguous(), th[e:e + 1].contiguous())
        assert torch.equal(Le[0], L[e]) and torch.equal(ge[0], g[e])
    h.close()


def test_argument_errors(dia):
    w = make_workload(0, n=64, m=5)
    R = _dev(w.R)
    with pytest.raises(dia.DiaError):
        dia.Handle(R, 4)                       # even m
    with pytest.raises(dia.DiaError):
        dia.Handle(R, 49)                      # above DIA_MAX_KERNEL_SIZE
    with pytest.raises(dia.DiaError):
        dia.Handle(R, 5, gain=0.0)
    h = dia.Handle(R, 5, sigma0=5.0)
    with pytest.raises(dia.DiaError):          # n_epochs > max_epochs
        h.eval_loss_grad(_dev(np.stack([w.I[0], w.I[0]])), _dev(np.stack([w.theta0[0]] * 2)))
    with pytest.raises(dia.DiaError):          # var given in MODEL mode
        h.eval_loss_grad(_dev(w.I), _dev(w.theta0), var=_dev(w.I))
    with pytest.raises(dia.DiaError):          # host tensor
        h.eval_loss_grad(torch.from_numpy(w.I), _dev(w.theta0))
    h.close()


def test_full_size_sampled_c4(dia):
    """BASELINE config 4 at full size in bench.py's launch configuration (4096^2, m = 19, batched
    epochs).  A sparse random mask (1 pixel in 256) makes the result a sum the oracle can afford
    pixel by pixel; the complementary-mask identity L(all) = L(mask) + L(~mask) ties the unmasked
    full-size evaluation to it."""
    E = 2
    w = make_workload(4, n_epochs=E)
    rng = np.random.default_rng(99)
    mask = (rng.random(w.I.shape) < 1.0 / 256).astype(np.uint8)
    h = _handle(dia, w)
    cfg = _ref_cfg(w)
    I = _dev(w.I)
    for name, th, kind in _points(w)[:2]:
        Lo, go, So = oracle.eval_loss_grad(cfg, w.R, w.I, th, mask=mask, want_scale=True)
        t = _dev(th)
        Lg, gg = h.eval_loss_grad(I, t, mask=_dev(mask))
        _compare(Lg, gg, Lo, go, So, kind, f"c4 full sampled {name}")
        if name == "P0":                       # gradient far from cancelling: FP32 strip rounding only
            La, ga = h.eval_loss_grad(I, t)
            Lc, gc = h.eval_loss_grad(I, t, mask=_dev(1 - mask))
            assert torch.allclose(La, Lg + Lc, rtol=1e-7, atol=0)
            assert float((ga - (gg + gc)).abs().max()) <= 2e-6 * float(ga.abs().max())
    h.close()


@pytest.mark.parametrize("c,E", [(2, 1), (3, 1), (4, 2)])
def test_full_size_direct(dia, c, E):
    """BASELINE configs 2, 3 and 4 at their full sizes (1024^2 Huber, 2048^2 flat + mask, 4096^2 batched -- the
    constant-bank launch bench.py times), every output against the oracle evaluated over all pixels (the
    OpenMP oracle needs about a second per 4096^2 epoch)."""
    w = make_workload(c, n_epochs=E)
    h = _handle(dia, w)
    cfg = _ref_cfg(w)
    I, mask = _dev(w.I), _dev(w.mask)
    for name, th, kind in _points(w)[:2]:
        Lo, go, So = oracle.eval_loss_grad(cfg, w.R, w.I, th, mask=w.mask, want_scale=True)
        Lg, gg = h.eval_loss_grad(I, _dev(th), mask=mask)
        _compare(Lg, gg, Lo, go, So, kind, f"c{c} full size {name}")
    h.close()


def test_row_bands_sum_to_the_full_image(dia):
    """the valid rows split into bands, each evaluated as an ordinary sub-image (its own handle, as a
    rank would); the band results add up to the full-image loss and gradient, and to the oracle's."""
    from paper_2104_13715_b200.sharding import row_band
    w = make_workload(4, n=300, n_epochs=1, m=19)
    th = w.theta_true.astype(np.float32)
    Lo, go, So = oracle.eval_loss_grad(_ref_cfg(w), w.R, w.I, th, want_scale=True)
    world = 3
    L = torch.zeros(1, dtype=torch.float64, device="cuda")
    g = torch.zeros((1, w.m * w.m + 1), dtype=torch.float64, device="cuda")
    for rank in range(world):
        v0, v1, i0, i1 = row_band(w.n, w.m, world, rank)
        h = dia.Handle(_dev(w.R[i0:i1]), w.m, sigma0=w.sigma0, gain=w.gain)
        Lb, gb = h.eval_loss_grad(_dev(w.I[:, i0:i1]), _dev(th))
        L += Lb
        g += gb
        h.close()
    _compare(L, g, Lo, go, So, "S", "row bands")
