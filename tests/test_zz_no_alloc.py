"""dia_eval_loss_grad_static: the allocation-free entry point (include/dia.h) against dia_eval_loss_grad on a handle.

Collected last on purpose (file name): the suite runs with pytest -x, and a failure here must not hide other tests.
The static entry point keeps its block partials in a file-scope __device__ array that every call shares and that keeps
the previous call's contents, so the test runs TWO calls in a row with different batches (the second smaller than the
first: stale partials of the first stay behind it in the array) and compares each with the existing path.  Both paths
launch the same kernel instantiation with the same grid here, so the results must be bit-identical; the assertion
also states the tolerance the GPU parity tests use (TOL = 1e-5 relative on the loss, e_norm on the gradient).
Passes alone in a fresh process and after the other GPU tests (it does not depend on what ran before: the set-up of
the static path is lazy and per device).
"""
import numpy as np
import pytest

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


def _both(dia, w, theta, E, mask=None, lam=0.0):
    """(loss, grad) of the first E epochs from the static entry point and from a handle with max_epochs == E."""
    huber = w.loss == "huber"
    kw = dict(loss=dia.LOSS_HUBER if huber else dia.LOSS_GAUSSIAN, sigma0=w.sigma0, gain=w.gain, lambda_reg=lam)
    R, I, th = _dev(w.R), _dev(w.I[:E]), _dev(theta[:E].astype(np.float32))
    mk = None if mask is None else _dev(mask[:E])
    flat = _dev(w.flat)
    np_ = w.m * w.m + 1
    Ls = torch.full((E,), float("nan"), dtype=torch.float64, device="cuda")
    gs = torch.full((E, np_), float("nan"), dtype=torch.float64, device="cuda")
    dia.dia_eval_loss_grad_static(w.n, w.n, w.m, R, E, I, mk, None, th, Ls, gs, d_flat=flat, **kw)
    h = dia.Handle(R, w.m, max_epochs=E, flat=flat, **kw)
    Lh, gh = h.eval_loss_grad(I, th, mask=mk)
    torch.cuda.synchronize()
    h.close()
    return (Ls.cpu(), gs.cpu()), (Lh.cpu(), gh.cpu())


def _assert_same(stat, hand):
    (Ls, gs), (Lh, gh) = stat, hand
    assert torch.isfinite(Ls).all() and torch.isfinite(gs).all()
    assert torch.allclose(Ls, Lh, rtol=TOL, atol=0)
    assert float((gs - gh).abs().max() / gh.abs().max()) <= TOL
    assert torch.equal(Ls, Lh) and torch.equal(gs, gh)          # same kernel, same grid, same orders


def test_static_entry_point_matches_the_handle_path_on_two_calls_in_a_row(dia):
    # 330 x 330, m = 9: 6 x 6 tiles per epoch with a ragged last row and column; rows not a multiple of 4 floats -> cp.async
    w = make_workload(2, n=330, m=9, n_epochs=3)                 # config 2: Huber loss
    first = _both(dia, w, w.theta0, 3)
    # second call: another theta, fewer epochs (a smaller part of the shared array), a mask (generic instantiation)
    rng = np.random.default_rng(5)
    mask = (rng.random(w.I.shape) > 0.02).astype(np.uint8)
    second = _both(dia, w, w.theta_true, 1, mask=mask, lam=10.0)
    _assert_same(*first)
    _assert_same(*second)
    assert not torch.equal(first[0][0][:1], second[0][0])


def test_static_entry_point_tma_path_and_size_limit(dia):
    w = make_workload(4, n=256, m=19, n_epochs=2)                # rows 16-byte aligned: TMA staging
    _assert_same(*_both(dia, w, w.theta0, 2))
    _assert_same(*_both(dia, w, w.theta_true, 2))
    # beyond the static array: 4096^2 at m = 19 is 296 columns of 362 doubles per epoch -> five epochs exceed 4 MiB.
    # Rejected on the host before anything is enqueued or dereferenced, so tiny stand-in tensors are enough here.
    assert 8 * 5 * 362 * 296 > dia.STATIC_SCRATCH_BYTES >= 8 * 4 * 362 * 296
    z = torch.zeros(16, dtype=torch.float32, device="cuda")
    o = torch.zeros(16, dtype=torch.float64, device="cuda")
    with pytest.raises(dia.DiaError, match="DIA_STATIC_SCRATCH_BYTES"):
        dia.dia_eval_loss_grad_static(4096, 4096, 19, z, 5, z, None, None, z, o, o, sigma0=5.0, gain=1.0)
