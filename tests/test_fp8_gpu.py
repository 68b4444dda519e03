"""FP8 (E4M3) operands (PAPER.md lines 382, 392 item 2; R19):
swiglu_mlp_fp8 through the C ABI against the fp64 FP8 oracle, element by element, same bound
as the bf16 path (the inputs are exact E4M3 values on both sides; products are exact, fp32
accumulation, one bf16 rounding): |y - y_ref| <= 2e-3 + 1.6e-2*|y_ref|."""
import numpy as np
import pytest
import torch

import oracle
from paper_2607_02521_b200 import binding as B
from paper_2607_02521_b200 import check, inputs

pytestmark = pytest.mark.gpu
ATOL, RTOL = 2e-3, 1.6e-2


def dev8(codes):
    return torch.from_numpy(np.ascontiguousarray(codes)).cuda()


def host(t):
    return t.view(torch.int16).cpu().numpy().view(np.uint16)


def run(A8, W1, W2, sg, su, variant=-1):
    M, N = A8.shape[0], W1.shape[0]
    dY = torch.full((M, N), float("nan"), dtype=torch.bfloat16, device="cuda")
    B.swiglu_mlp_fp8(dev8(A8), dev8(W1), dev8(W2), dY, sg, su, variant)
    torch.cuda.synchronize()
    return host(dY)


def assert_parity(y_bits, y_ref, what):
    rep = check.compare(y_bits, y_ref)
    y = inputs.bf16_bits_to_f64(y_bits)
    assert np.all(np.isfinite(y)), what
    assert np.all(np.abs(y - y_ref) <= ATOL + RTOL * np.abs(y_ref)), (what, rep)
    return rep


SHAPES = [(1, 128, 128), (7, 136, 80), (16, 4864, 896), (33, 264, 208), (100, 1160, 336),
          (128, 4864, 896), (129, 264, 208), (300, 1160, 336), (513, 392, 1104), (2560, 1032, 144)]


@pytest.mark.parametrize("variant", [-1, 0, 1, 2, 3, 4])
@pytest.mark.parametrize("M,N,K", SHAPES)
def test_fp8_every_variant_on_odd_shapes(variant, M, N, K):
    if variant == 2 and M > 128:
        pytest.skip("small-M variant handles M <= 128")
    A8, W1, W2, sg, su = inputs.make_fp8_case(M, N, K, seed=2000 + M + N + K, std=0.05)
    y_ref, _ = oracle.swiglu_oracle_fp8(A8, W1, W2, sg, su)
    assert_parity(run(A8, W1, W2, sg, su, variant), y_ref, ("fp8", variant, M, N, K))


@pytest.mark.parametrize("ksplit", [1, 2, 3, 5, 8])
def test_fp8_small_m_every_cluster_size(ksplit, monkeypatch):
    monkeypatch.setenv("SWIGLU_KSPLIT", str(ksplit))
    B.swiglu_reload_env()
    try:
        for M in (1, 16, 40, 128):
            A8, W1, W2, sg, su = inputs.make_fp8_case(M, 520, 1424, seed=2100 + M, std=0.05)
            y_ref, _ = oracle.swiglu_oracle_fp8(A8, W1, W2, sg, su)
            assert_parity(run(A8, W1, W2, sg, su, 2), y_ref, ("fp8 smallm", M, ksplit))
    finally:
        monkeypatch.delenv("SWIGLU_KSPLIT")
        B.swiglu_reload_env()


def test_fp8_scales_and_special_values():
    """Scales far from 1 (Gate spans both SiLU tails), exact zeros, the largest finite code."""
    M, N, K = 64, 392, 336
    A8, W1, W2, _, _ = inputs.make_fp8_case(M, N, K, seed=2200)
    A8[0, :] = 0x00                        # a zero row: Y row must be exactly +-0
    A8[1, :16] = 0x7E                      # 448
    W1[0, :16] = 0xFE                      # -448
    for sg, su in ((0.004, 0.5), (0.25, 1e-3), (1.0 / 64, 1.0 / 64)):
        y_ref, _ = oracle.swiglu_oracle_fp8(A8, W1, W2, sg, su)
        y = run(A8, W1, W2, sg, su)
        assert_parity(y, y_ref, ("fp8 scales", sg, su))
        assert np.all((y[0] & 0x7FFF) == 0)


def test_fp8_baseline_shapes_sampled_rows_and_determinism():
    """The 1.5B and 7B BASELINE.json shapes with FP8 operands at every M of the config, automatic
    dispatch, rows of every row tile; run-to-run bitwise determinism."""
    for shape in ("qwen2.5-1.5b", "qwen2.5-7b"):
        K, N, seed, Ms = inputs.SHAPES[shape]
        A8, W1, W2, sg, su = inputs.make_fp8_case(max(Ms), N, K, seed=2300 + seed)
        dW1, dW2 = dev8(W1), dev8(W2)
        for M in Ms:
            rows = inputs.sample_rows(M)
            if len(rows) > 64:
                rows = rows[np.linspace(0, len(rows) - 1, 64).round().astype(int)]
            y_ref, _ = oracle.swiglu_oracle_fp8(A8[:M], W1, W2, sg, su, rows=rows)
            dA = dev8(A8[:M])
            outs = []
            for _ in range(2):
                dY = torch.full((M, N), float("nan"), dtype=torch.bfloat16, device="cuda")
                B.swiglu_mlp_fp8(dA, dW1, dW2, dY, sg, su)
                torch.cuda.synchronize()
                assert bool(torch.isfinite(dY.float()).all()), (shape, M)
                outs.append(host(dY))
            assert np.array_equal(outs[0], outs[1])
            rep = check.compare(outs[0][rows], y_ref)
            assert rep.mismatches == 0, (shape, M, rep)


def test_fp8_argument_validation():
    M, N, K = 16, 136, 80
    A8, W1, W2, sg, su = inputs.make_fp8_case(M, N, K, seed=2400)
    dY = torch.zeros((M, N), dtype=torch.bfloat16, device="cuda")
    lib = B.load()
    a, w1, w2 = dev8(A8), dev8(W1), dev8(W2)
    args = (a.data_ptr(), w1.data_ptr(), w2.data_ptr(), dY.data_ptr())
    assert lib.swiglu_mlp_fp8(*args, M, N, 72, 1.0, 1.0, None) == B.SWIGLU_ERR_UNSUPPORTED   # K % 16
    assert lib.swiglu_mlp_fp8(*args, M, 132, K, 1.0, 1.0, None) == B.SWIGLU_ERR_UNSUPPORTED  # N % 8
    assert lib.swiglu_mlp_fp8(*args, -1, N, K, 1.0, 1.0, None) == B.SWIGLU_ERR_BAD_SHAPE
    assert lib.swiglu_mlp_fp8(None, args[1], args[2], args[3], M, N, K, 1.0, 1.0, None) == B.SWIGLU_ERR_NULL_POINTER
    assert lib.swiglu_mlp_fp8(args[0], args[1], args[2], args[0], M, N, K, 1.0, 1.0, None) == B.SWIGLU_ERR_ALIASING
    assert lib.swiglu_mlp_fp8(*args, M, N, K, float("nan"), 1.0, None) == B.SWIGLU_ERR_UNSUPPORTED
    assert lib.swiglu_mlp_fp8(*args, 0, N, K, 1.0, 1.0, None) == B.SWIGLU_OK
    assert lib.swiglu_mlp_fp8_ex(*args, M, N, K, 1.0, 1.0, 9, None) == B.SWIGLU_ERR_UNSUPPORTED
