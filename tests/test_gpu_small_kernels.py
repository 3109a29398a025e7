"""GPU-vs-oracle parity of the register-resident kernel for small kernels (m = 1, 3, 5; dia_eval_small.cuh), which
evaluates the plain objective (no mask / flat / variance map / background polynomial) of handles with m <= 5.

Same protocol as tests/test_gpu_parity.py (loss to 1e-5 relative, gradient to 1e-5 of the cancellation-free scale S_p),
on shapes chosen for this kernel's geometry: 8-pixel strips, lanes side by side up to 256 columns, 2-16 rows per thread,
128-bit loads when rows are 16-byte aligned and scalar loads when not.
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


def _dev(a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda().contiguous()


def _compare(Lg, gg, Lo, go, So, kind, tag):
    Lg, gg = Lg.cpu().numpy(), gg.cpu().numpy()
    for e in range(Lo.shape[0]):
        d = np.abs(gg[e] - go[e])
        e_norm, e_S = d.max() / np.abs(go[e]).max(), (d / So[e]).max()
        print(f"{tag} e{e}: dL/L={abs(Lg[e]-Lo[e])/abs(Lo[e]):.2e} e_norm={e_norm:.2e} e_S={e_S:.2e}")
        assert abs(Lg[e] - Lo[e]) <= TOL * abs(Lo[e]), f"{tag} epoch {e}: loss {Lg[e]} vs {Lo[e]}"
        assert e_S <= TOL, f"{tag} epoch {e}: e_S = {e_S:.3e}"
        if kind == "norm":
            assert e_norm <= TOL, f"{tag} epoch {e}: e_norm = {e_norm:.3e}"


def _crop(w, nr, nc):
    return np.ascontiguousarray(w.R[:nr, :nc]), np.ascontiguousarray(w.I[:, :nr, :nc])


SHAPES = [  # (rows, cols): what it exercises
    (300, 300),    # 128-bit loads; two tiles across (256-pixel warps), ragged right and bottom edges
    (333, 333),    # rows not 16-byte aligned: scalar loads
    (97, 700),     # wide and flat: three tiles across, few rows
    (500, 20),     # narrow: four lanes side by side, eight stacked
    (64, 262),     # valid width 256 + a few pixels at m = 5: a second tile column with one or two strips
]


@pytest.mark.parametrize("loss", ["gaussian", "huber"])
@pytest.mark.parametrize("m", [1, 3, 5])
@pytest.mark.parametrize("nr,nc", SHAPES)
def test_small_kernel_parity(dia, nr, nc, m, loss):
    w = make_workload(2 if loss == "huber" else 4, n=max(nr, nc), m=m, n_epochs=2)
    R, I = _crop(w, nr, nc)
    kw = dict(sigma0=w.sigma0, gain=w.gain)
    cfg = oracle.RefConfig(nr, nc, m, loss=oracle.LOSS_HUBER if loss == "huber" else oracle.LOSS_GAUSSIAN, **kw)
    h = dia.Handle(_dev(R), m, max_epochs=2, loss=dia.LOSS_HUBER if loss == "huber" else dia.LOSS_GAUSSIAN, **kw)
    for th, kind in ((w.theta0, "norm"), (w.theta_true.astype(np.float32), "S")):
        Lo, go, So = oracle.eval_loss_grad(cfg, R, I, th, want_scale=True)
        Lg, gg = h.eval_loss_grad(_dev(I), _dev(th))
        Lg2, gg2 = h.eval_loss_grad(_dev(I), _dev(th))
        assert torch.equal(Lg, Lg2) and torch.equal(gg, gg2), "evaluation is not deterministic"
        _compare(Lg, gg, Lo, go, So, kind, f"small m={m} {nr}x{nc} {loss}")
    h.close()


@pytest.mark.parametrize("m", [1, 3, 5])
def test_small_kernel_is_the_one_that_runs_and_agrees_with_the_generic_kernel(dia, monkeypatch, m):
    """DIA_DISABLE_SMALL=1 forces the generic shared-memory kernel: both must agree with the oracle, and with each other
    far inside the tolerance; a mask (generic kernel on the same handle) of all ones gives the generic result."""
    w = make_workload(4, n=400, m=m, n_epochs=3)
    cfg = oracle.RefConfig(w.n, w.n, m, sigma0=w.sigma0, gain=w.gain)
    th = w.theta_true.astype(np.float32)
    Lo, go, So = oracle.eval_loss_grad(cfg, w.R, w.I, th, want_scale=True)
    h = dia.Handle(_dev(w.R), m, max_epochs=3, sigma0=w.sigma0, gain=w.gain)
    Ls, gs = h.eval_loss_grad(_dev(w.I), _dev(th))
    Lm, gm = h.eval_loss_grad(_dev(w.I), _dev(th), mask=_dev(np.ones(w.I.shape, np.uint8)))
    h.close()
    monkeypatch.setenv("DIA_DISABLE_SMALL", "1")
    h2 = dia.Handle(_dev(w.R), m, max_epochs=3, sigma0=w.sigma0, gain=w.gain)
    Lg, gg = h2.eval_loss_grad(_dev(w.I), _dev(th))
    h2.close()
    _compare(Ls, gs, Lo, go, So, "S", f"small m={m}")
    _compare(Lg, gg, Lo, go, So, "S", f"generic m={m}")
    assert not (torch.equal(gs, gg) and torch.equal(Ls, Lg)), "the small kernel did not run (same bits as the generic one)"
    assert (Ls - Lg).abs().max() <= 1e-6 * Lg.abs().max()
    assert ((gs - gg).abs().cpu().numpy() / So).max() <= 5e-6
    assert (Lm - Lg).abs().max() <= 1e-6 * Lg.abs().max()


@pytest.mark.parametrize("m", [1, 3, 5])
def test_small_kernel_right_edge_positions(dia, monkeypatch, m):
    """The ragged right edge, lane by lane.  A warp's 32 strips of 8 pixels either all take the unpredicated path or all
    the predicated one, and the last strip may hold 1 .. 8 valid pixels: widths are chosen so that the edge falls into
    the first, a middle and the last lane of a warp, in the first and in a later tile column, with 16-byte aligned rows
    (128-bit loads) and without.  Several tile rows on three CTAs, so that the rotation of the tile columns by the tile
    row meets every column.  Against the oracle at the parity tolerance, and against the generic kernel on the same data
    (DIA_DISABLE_SMALL=1) far inside it; both deterministic."""
    widths = [16, 20, 36, 132, 136, 140, 250, 256, 260, 264, 268, 508, 512, 516, 520, 772, 1028, 333, 262, 515]
    rows = 150
    w = make_workload(4, n=1028, m=m, n_epochs=2)
    th = w.theta_true.astype(np.float32)
    res = {}
    for disable in ("0", "1"):
        monkeypatch.setenv("DIA_DISABLE_SMALL", disable)
        monkeypatch.setenv("DIA_GRID_LIMIT", "3")
        for nc in widths:
            R, I = _crop(w, rows, nc)
            h = dia.Handle(_dev(R), m, max_epochs=2, sigma0=w.sigma0, gain=w.gain)
            L, g = h.eval_loss_grad(_dev(I), _dev(th))
            L2, g2 = h.eval_loss_grad(_dev(I), _dev(th))
            assert torch.equal(L, L2) and torch.equal(g, g2), f"width {nc}: evaluation is not deterministic"
            res[(disable, nc)] = (L.cpu().numpy(), g.cpu().numpy())
            h.close()
    for nc in widths:
        (Ls, gs), (Lg, gg) = res[("0", nc)], res[("1", nc)]
        R, I = _crop(w, rows, nc)
        cfg = oracle.RefConfig(rows, nc, m, sigma0=w.sigma0, gain=w.gain)
        Lo, go, So = oracle.eval_loss_grad(cfg, R, I, th, want_scale=True)
        _compare(torch.from_numpy(Ls), torch.from_numpy(gs), Lo, go, So, "S", f"small m={m} width {nc}")
        assert np.abs(Ls - Lg).max() <= 1e-6 * np.abs(Lg).max(), f"width {nc}: loss {Ls} vs {Lg}"
        assert (np.abs(gs - gg) / So).max() <= 5e-6, f"width {nc}: small and generic kernel differ by {(np.abs(gs - gg) / So).max():.3e} of S"


@pytest.mark.parametrize("grid_limit", [1, 3])
def test_small_kernel_many_tiles_per_cta_batched_and_singles(dia, monkeypatch, grid_limit):
    """One or three CTAs walk through every (epoch, tile) item: epoch changes inside a CTA, partial columns shared by
    many tiles.  Batched == singles bit for bit (the image is cut the same way whatever the batch size)."""
    monkeypatch.setenv("DIA_GRID_LIMIT", str(grid_limit))
    w = make_workload(4, n=520, m=3, n_epochs=3)
    cfg = oracle.RefConfig(w.n, w.n, 3, sigma0=w.sigma0, gain=w.gain)
    h = dia.Handle(_dev(w.R), 3, max_epochs=3, sigma0=w.sigma0, gain=w.gain)
    th = w.theta_true.astype(np.float32)
    Lo, go, So = oracle.eval_loss_grad(cfg, w.R, w.I, th, want_scale=True)
    I, tht = _dev(w.I), _dev(th)
    L, g = h.eval_loss_grad(I, tht)
    _compare(L, g, Lo, go, So, "S", f"small grid={grid_limit}")
    for e in range(3):
        Le, ge = h.eval_loss_grad(I[e:e + 1].contiguous(), tht[e:e + 1].contiguous())
        assert torch.equal(Le[0], L[e]) and torch.equal(ge[0], g[e])
    h.close()


def test_small_kernel_unpoisoned_by_border_and_minimum_size(dia):
    """NaN in the border of I (outside the valid set) must not reach a result; n == m leaves one valid pixel."""
    w = make_workload(0, n=128, m=3)
    h = dia.Handle(_dev(w.R), 3, sigma0=w.sigma0, gain=w.gain)
    th = _dev(w.theta_true.astype(np.float32))
    L0, g0 = h.eval_loss_grad(_dev(w.I), th)
    Ip = w.I.copy()
    Ip[:, :1, :] = np.nan; Ip[:, -1:, :] = np.nan; Ip[:, :, :1] = np.nan; Ip[:, :, -1:] = np.nan
    L1, g1 = h.eval_loss_grad(_dev(Ip), th)
    assert torch.equal(L0, L1) and torch.equal(g0, g1)
    h.close()
    rng = np.random.default_rng(2)
    for m in (1, 3, 5):
        R = (100 + 50 * rng.random((m, m))).astype(np.float32)
        I = (120 + 50 * rng.random((1, m, m))).astype(np.float32)
        th = np.concatenate([np.full(m * m, 1.0 / (m * m)), [2.0]]).astype(np.float32)
        cfg = oracle.RefConfig(m, m, m, sigma0=3.0, gain=1.5)
        Lo, go, So = oracle.eval_loss_grad(cfg, R, I, th, want_scale=True)
        h = dia.Handle(_dev(R), m, sigma0=3.0, gain=1.5)
        Lg, gg = h.eval_loss_grad(_dev(I), _dev(th))
        _compare(Lg, gg, Lo, go, So, "norm", f"n==m=={m}")
        h.close()


def test_small_kernel_one_reference_per_epoch_and_fit(dia):
    """n_refs == max_epochs (a batch of independent stamps) through the small kernel, and a lock-step fit (the kernel
    inside the CUDA-graph loop, done flags included) against the oracle: fitted K, B0 and P to 1e-4."""
    m, E = 3, 5
    w = make_workload(0, n=142, m=m, n_epochs=E)
    Rs = np.stack([np.roll(w.R, 7 * e, axis=1) for e in range(E)])      # a different reference per epoch
    Is = w.I
    kw = dict(sigma0=w.sigma0, gain=w.gain)
    h = dia.Handle(_dev(Rs), m, max_epochs=E, **kw)
    cfg = oracle.RefConfig(142, 142, m, **kw)
    th = w.theta_true.astype(np.float32)
    Lg, gg = h.eval_loss_grad(_dev(Is), _dev(th))
    for e in range(E):
        Lo, go, So = oracle.eval_loss_grad(cfg, Rs[e], Is[e:e + 1], th[e:e + 1], want_scale=True)
        _compare(Lg[e:e + 1], gg[e:e + 1], Lo, go, So, "S", f"small stamps e{e}")
    h.close()
    # lock-step fit on a shared reference
    h = dia.Handle(_dev(w.R), m, max_epochs=E, **kw)
    fo = dict(force_adam_iters=25, force_lbfgs_iters=8)
    thg, rg = h.fit(_dev(w.I), _dev(w.theta0), dia.FitOpts.default(**fo))
    tho, ro = oracle.fit(cfg, w.R, w.I, w.theta0, oracle.RefFitOpts.default(**fo))
    thg = thg.cpu().numpy()
    for e in range(E):
        assert rg[e].n_evals == ro[e].n_evals
        assert np.abs(thg[e][:-1] - tho[e][:-1]).max() <= 1e-4 * np.abs(tho[e][:-1]).max()
        assert abs(thg[e][-1] - tho[e][-1]) <= 1e-4 * max(abs(tho[e][-1]), 1.0)
        assert abs(rg[e].photometric_scale - ro[e].photometric_scale) <= 1e-4 * abs(ro[e].photometric_scale)
    # a free-running batch: epochs stop at different iterations (done flags skip them), same result as singles
    thb, rb = h.fit(_dev(w.I), _dev(w.theta0), dia.FitOpts.default())
    for e in range(E):
        th1, r1 = h.fit(_dev(w.I[e:e + 1]), _dev(w.theta0[e:e + 1]), dia.FitOpts.default())
        assert r1[0].n_evals == rb[e].n_evals and torch.equal(th1[0], thb[e])
    h.close()


@pytest.mark.parametrize("m", [1, 3])
def test_small_kernel_full_size_c4(dia, m):
    """The 4096^2 field of BASELINE config 4, two epochs, in the launch configuration bench.py's small-kernel leg and
    sweep time (16 rows per thread, 444 or 296 CTAs, 128-bit loads): every output against the oracle over all pixels."""
    w = make_workload(4, m=m, n_epochs=2)
    cfg = oracle.RefConfig(w.n, w.n, m, sigma0=w.sigma0, gain=w.gain)
    h = dia.Handle(_dev(w.R), m, max_epochs=16, sigma0=w.sigma0, gain=w.gain)     # a 16-epoch handle cuts 16-row strips
    I = _dev(w.I)
    for th, kind in ((w.theta0, "norm"), (w.theta_true.astype(np.float32), "S")):
        Lo, go, So = oracle.eval_loss_grad(cfg, w.R, w.I, th, want_scale=True)
        Lg, gg = h.eval_loss_grad(I, _dev(th))
        _compare(Lg, gg, Lo, go, So, kind, f"small m={m} c4 full size")
    h.close()
