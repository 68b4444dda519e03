"""Pins of the FP8 (E4M3) oracle (oracle.swiglu_oracle_fp8; PAPER.md lines 382, 392 item 2;
DESIGN.md R19) and of the E4M3 input quantiser in inputs.py."""
from fractions import Fraction

import numpy as np
import pytest
import torch

import oracle
from paper_2607_02521_b200 import inputs


def test_decode_closed_forms():
    """Values fixed by the OCP FP8 specification (E4M3: bias 7, max 448, min subnormal 2^-9)."""
    f = oracle.e4m3_to_f64
    assert f(0x00) == 0.0 and f(0x80) == 0.0 and np.signbit(f(0x80))
    assert f(0x38) == 1.0 and f(0xB8) == -1.0
    assert f(0x01) == 2.0 ** -9 and f(0x07) == 7 * 2.0 ** -9
    assert f(0x08) == 2.0 ** -6                       # smallest normal
    assert f(0x7E) == 448.0 and f(0xFE) == -448.0     # largest finite
    assert f(0x40) == 2.0 and f(0x3C) == 1.5 and f(0x30) == 0.5
    assert np.isnan(f(0x7F)) and np.isnan(f(0xFF))    # no infinities in e4m3fn


def test_decode_matches_the_library_for_all_256_codes():
    codes = np.arange(256, dtype=np.uint8)
    lib = torch.from_numpy(codes).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    ours = np.array([oracle.e4m3_to_f64(int(c)) for c in codes])
    assert np.array_equal(np.isnan(lib), np.isnan(ours))
    ok = ~np.isnan(lib)
    assert np.array_equal(lib[ok], ours[ok])
    assert np.array_equal(np.signbit(lib[ok]), np.signbit(ours[ok]))


def test_input_quantiser_matches_the_library_rounding():
    rng = np.random.Generator(np.random.Philox(key=5))
    x = np.concatenate([rng.standard_normal(20000).astype(np.float32) * s for s in (1e-3, 0.05, 1, 30, 300)])
    x = np.concatenate([x, np.float32([0.0, -0.0, 448.0, 449.0, 1e9, -1e9, 2.0 ** -10, 3 * 2.0 ** -10,
                                       1.0625, 1.1875, 2.0 ** -9, 464.0, 479.0])])
    ours = inputs.f32_to_e4m3_bits(x)
    lib = torch.from_numpy(x).clamp(-448, 448).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    assert np.array_equal(ours, lib)


@pytest.mark.parametrize("M,N,K", [(1, 1, 1), (2, 3, 5), (3, 8, 17), (5, 2, 16)])
def test_brute_force_exact_rationals(M, N, K):
    A8, W1, W2, _, _ = inputs.make_fp8_case(M, N, K, seed=7 + M + N + K)
    sg, su = 0.5, 0.25                                 # exact binary scales
    y, _ = oracle.swiglu_oracle_fp8(A8, W1, W2, sg, su)
    dec = lambda b: Fraction(oracle.e4m3_to_f64(int(b)))
    for m in range(M):
        for n in range(N):
            g = sum(dec(A8[m, k]) * dec(W1[n, k]) for k in range(K)) * Fraction(sg)
            u = sum(dec(A8[m, k]) * dec(W2[n, k]) for k in range(K)) * Fraction(su)
            want = oracle.silu(float(g)) * float(u)
            assert y[m, n] == pytest.approx(want, rel=1e-14, abs=1e-300)


def test_equals_the_bf16_oracle_on_the_same_values():
    """Every E4M3 value is exactly representable in bf16, so with unit scales the FP8 oracle must
    reproduce the (separately pinned) bf16 oracle on the converted inputs, weights transposed
    to its [K,N] layout -- bit for bit, since both sum k ascending in fp64."""
    M, N, K = 7, 40, 96
    A8, W1, W2, _, _ = inputs.make_fp8_case(M, N, K, seed=21)
    to_bf16 = lambda c: inputs.f64_to_bf16_bits_exact(
        np.vectorize(oracle.e4m3_to_f64)(c.astype(np.uint8)).astype(np.float64))
    y8, _ = oracle.swiglu_oracle_fp8(A8, W1, W2, 1.0, 1.0)
    y16, _ = oracle.swiglu_oracle(to_bf16(A8), np.ascontiguousarray(to_bf16(W1).T),
                                  np.ascontiguousarray(to_bf16(W2).T))
    assert np.array_equal(y8, y16)
    rows = [5, 0, 3]
    ysub, _ = oracle.swiglu_oracle_fp8(A8, W1, W2, 1.0, 1.0, rows=rows)
    assert np.array_equal(ysub, y8[rows])


def test_scales_enter_before_the_activation_for_gate_and_linearly_for_up():
    M, N, K = 4, 24, 64
    A8, W1, W2, _, _ = inputs.make_fp8_case(M, N, K, seed=22)
    dec = np.vectorize(oracle.e4m3_to_f64)
    G = dec(A8) @ dec(W1).T                            # library fp64 matmuls
    U = dec(A8) @ dec(W2).T
    sg, su = 0.02, 0.03
    y, _ = oracle.swiglu_oracle_fp8(A8, W1, W2, sg, su)
    want = np.vectorize(oracle.silu)(sg * G) * (su * U)
    assert np.allclose(y, want, rtol=1e-12, atol=1e-15)
    y2, _ = oracle.swiglu_oracle_fp8(A8, W1, W2, sg, 2 * su)
    assert np.array_equal(y2, 2 * y)                   # Up scale is linear, exactly
    y3, _ = oracle.swiglu_oracle_fp8(A8, W1, W2, 2 * sg, su)
    assert not np.allclose(y3, 2 * y)                  # Gate scale is inside SiLU
