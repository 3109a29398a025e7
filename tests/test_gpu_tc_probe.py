"""What dia_hessian's tensor-core kernel (csrc/dia_hess_tc.cuh) rests on, measured with the one-CTA probe
dia_tc_probe_gemm (csrc/dia_tc_probe.cuh; same operand layout, descriptors and hi / lo split, ONE accumulation chain
over all of K):
  * the shared-memory layout and the descriptors are right: integer data give the exact product, for every N;
  * tcgen05.mma adds each product to the float32 accumulator after aligning it to the larger exponent and TRUNCATING it
    below 2^-25 of that exponent -- it never rounds up, and addends below that threshold vanish however many there are.
    This is why the kernel keeps a chain to one tile row (64 pixels) and sums the rows in registers and FP64;
  * accordingly the error of a split-float16 sum of positive terms is a BIAS that grows with the chain length.
These are statements about the hardware (B200, sm_100a); should a later part behave differently the numbers printed here
say how.  python -m pytest -m gpu -s tests/test_gpu_tc_probe.py prints the tables quoted in profiles/r02_tc_hessian.md.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

ULP = 2.0 ** -23        # of 1.0


@pytest.fixture(scope="module")
def dia():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    import paper_2104_13715_b200 as dia
    dia.load_library()
    return dia


def _run(dia, A, B, mode):
    D = dia.dia_tc_probe_gemm(torch.from_numpy(A.astype(np.float32)).cuda(), torch.from_numpy(B.astype(np.float32)).cuda(), mode)
    torch.cuda.synchronize()
    return D.cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("mode", [0, 1, 2, 3])
@pytest.mark.parametrize("N", [32, 64, 128, 192, 256])
def test_layout_and_descriptors_exact_on_integer_data(dia, mode, N):
    rng = np.random.default_rng(10 * N + mode)
    K = 192
    A = rng.integers(-3, 4, (128, K)).astype(np.float64)
    B = rng.integers(-2, 3, (N, K)).astype(np.float64)
    assert np.array_equal(_run(dia, A, B, mode), A @ B.T)


@pytest.mark.parametrize("mode", [0, 2])
def test_accumulator_truncates_addends_below_2_pow_minus_25(dia, mode):
    """Accumulator 1.0 (first instruction), then T = 64 instructions that each add KS equal products of 2^-e (columns
    with odd n: 1.5 x 2^-e)."""
    KS, T, N = (16, 64, 64) if mode == 0 else (8, 64, 64)
    K = 64 * -(-(KS * (1 + T)) // 64)
    rows = []
    for e in range(23, 31):
        A = np.zeros((128, K))
        B = np.zeros((N, K))
        A[:, 0] = 1.0
        B[:, 0] = 1.0
        A[:, KS:KS * (1 + T)] = 2.0 ** -12
        B[:, KS:KS * (1 + T)] = 2.0 ** (12 - e)
        B[1::2, KS:KS * (1 + T)] *= 1.5
        D = _run(dia, A, B, mode)
        assert np.all(D == D[0:1, :]) and np.all(D[:, 0::2] == D[0, 0]) and np.all(D[:, 1::2] == D[0, 1])
        exact = np.array([T * KS * 2.0 ** -e, 1.5 * T * KS * 2.0 ** -e]) / ULP
        got = (D[0, :2] - 1.0) / ULP
        rows.append((e, 2.0 ** -e / ULP, exact, got))
        print(f"mode {mode}: product = {2.0 ** -e / ULP:.4f} ulp (x1.5 odd n), {T} x {KS} of them: exact +{exact[0]:.0f} / +{exact[1]:.0f} ulp, "
              f"tensor core +{got[0]:.0f} / +{got[1]:.0f} ulp")
    for e, p_ulp, exact, got in rows:
        assert np.all(got <= exact)                       # never rounds up
        if p_ulp >= 0.5:                                   # products of at least 2^-24: on the accumulator's grid or kept
            assert got[0] == exact[0]
        if p_ulp * 1.5 < 0.25:                             # below 2^-25 of the accumulator: gone, all T x KS of them
            assert got[0] == 0.0 and got[1] == 0.0
    e25 = [r for r in rows if r[0] == 25][0]
    assert e25[3][0] == e25[2][0]                          # 0.25 ulp products are kept exactly ...
    assert e25[3][1] == e25[2][0]                          # ... and 0.375 ulp products are cut to 0.25 ulp: truncation at 2^-25


def test_split_float16_sum_bias_grows_with_the_chain(dia):
    """Sky-like positive data (1000 +- 30 times weights near 1): relative error of the split-float16 sums against
    FP64, one chain over K pixels."""
    rng = np.random.default_rng(4)
    out = {}
    for K in (64, 256, 1024, 4096):
        A = 1000.0 + 30.0 * rng.uniform(-1, 1, (128, K))
        B = (1000.0 + 30.0 * rng.uniform(-1, 1, (128, K))) * 1e-3
        A32, B32 = A.astype(np.float32).astype(np.float64), B.astype(np.float32).astype(np.float64)
        rel = (_run(dia, A32, B32, 1) - A32 @ B32.T) / (A32 @ B32.T)
        out[K] = (rel.mean(), np.abs(rel).max())
        print(f"split float16, chain of {K} pixels: mean relative error {rel.mean():+.2e}, max {np.abs(rel).max():.2e}")
    assert abs(out[64][0]) <= 1.5e-7 and out[64][1] <= 1e-6          # one tile row: what the kernel does
    assert out[4096][0] <= -1e-6                                     # a long chain is systematically LOW
    assert out[4096][0] < out[1024][0] < out[256][0] < 0.0
