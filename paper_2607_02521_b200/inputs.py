"""Seeded synthetic inputs shared by the tests, the bench and smoke().

This module holds NONE of the method's arithmetic (no matmul, no SiLU): it only draws
random numbers, rounds them to bf16 bit patterns and names the workload shapes.  It is the
one module both the CUDA-path harness and the oracle's tests may use (the oracle itself
imports nothing from here).

Workload recipe ("we construct random BF16
input tensors A and weight matrices W1, W2 matching each model's dimensions";
BASELINE.json configs: A ~ N(0,1), W1, W2 ~ N(0, 0.02) read as std 0.02):

* generator: numpy Philox (counter-based), key = 4*seed + stream, stream 0 = W1, 1 = W2,
  2 = A; values drawn row-major in fp32, scaled, rounded to bf16 round-to-nearest-even;
* one seed per shape (0.5B -> 0 ... 72B -> 4); A for batch M is the first M rows of the
  stream, so A(M) is a prefix of A(M') for M < M'.
"""
from __future__ import annotations

import numpy as np

# name -> (K, N, seed, M values)  -- BASELINE.json configs[0..4]
SHAPES = {
    "qwen2.5-0.5b": (896, 4864, 0, (16,)),
    "qwen2.5-1.5b": (1536, 8960, 1, (1, 16, 128, 1024, 4096)),
    "qwen2.5-7b": (3584, 18944, 2, (1, 16, 128, 1024, 4096)),
    "qwen2.5-32b": (5120, 27648, 3, (1, 16, 128, 1024, 4096)),
    "qwen2.5-72b": (8192, 29568, 4, (1, 16, 128, 1024, 4096, 8192)),
}
# The paper's own grid (Table 1 and section 4.2); seeds continue.
PAPER_SHAPES = {
    "paper-0.5b": (896, 4864, 10, (256, 512, 1024, 2048, 4096)),
    "paper-1.5b": (1536, 8960, 11, (256, 512, 1024, 2048, 4096)),
    "paper-14b": (5120, 13824, 12, (256, 512, 1024, 2048, 4096)),
    "paper-72b": (8192, 29568, 13, (256, 512, 1024, 2048, 4096)),
}
W_STD = 0.02
_CHUNK = 1 << 24  # elements per generation chunk (bounds the fp32 scratch to 64 MiB)


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """fp32 -> bf16 bit pattern (uint16), round-to-nearest-even.  Finite inputs only."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = (u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))) >> np.uint32(16)
    return r.astype(np.uint16)


def bf16_bits_to_f64(bits: np.ndarray) -> np.ndarray:
    """bf16 bit pattern (uint16) -> fp64, exact."""
    b = np.ascontiguousarray(bits, dtype=np.uint16)
    return (b.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)


def f64_to_bf16_bits_exact(x) -> np.ndarray:
    """For hand-written test matrices whose entries are exactly representable in bf16."""
    x = np.asarray(x, dtype=np.float64)
    bits = f32_to_bf16_bits(x.astype(np.float32))
    if not np.array_equal(bf16_bits_to_f64(bits), x):
        raise ValueError("entries are not exactly representable in bf16")
    return bits


def _normal_bits(key: int, count: int, scale: float) -> np.ndarray:
    gen = np.random.Generator(np.random.Philox(key=int(key)))
    out = np.empty(count, dtype=np.uint16)
    for lo in range(0, count, _CHUNK):
        n = min(_CHUNK, count - lo)
        v = gen.standard_normal(n, dtype=np.float32)
        if scale != 1.0:
            v *= np.float32(scale)
        out[lo:lo + n] = f32_to_bf16_bits(v)
    return out


def make_weights(K: int, N: int, seed: int, std: float = W_STD):
    """(W1, W2) bf16 bit patterns, each [K, N] row-major, ~ N(0, std)."""
    w1 = _normal_bits(4 * seed + 0, K * N, std).reshape(K, N)
    w2 = _normal_bits(4 * seed + 1, K * N, std).reshape(K, N)
    return w1, w2


def make_activations(M: int, K: int, seed: int):
    """A bf16 bit patterns [M, K] row-major, ~ N(0, 1); a prefix of the seed's A stream."""
    return _normal_bits(4 * seed + 2, M * K, 1.0).reshape(M, K)


def make_case(M: int, N: int, K: int, seed: int, std: float = W_STD):
    """(A, W1, W2) for an arbitrary parity-test shape."""
    w1, w2 = make_weights(K, N, seed, std)
    return make_activations(M, K, seed), w1, w2


def sample_rows(M: int, per_tile: int = 8, tile: int = 128):
    """Row sample for full-size parity: in every 128-row tile the in-tile offsets
    {0,31,32,63,64,95,96,127} (both ends of every 32-lane TMEM quarter), clipped to M."""
    offs = (0, 31, 32, 63, 64, 95, 96, 127)[:per_tile]
    rows = sorted({t + o for t in range(0, M, tile) for o in offs if t + o < M} | {M - 1})
    return np.asarray(rows, dtype=np.int64)


# ---------------------------------------------------------------------------------------
# FP8 (OCP E4M3, "e4m3fn") inputs for the FP8-operand entry point.
# Input preparation only: quantising random numbers to the format the call consumes.
# ---------------------------------------------------------------------------------------
def _e4m3_magnitudes() -> np.ndarray:
    """The 127 finite non-negative E4M3 values in code order (code = index)."""
    code = np.arange(127)
    e, m = code >> 3, code & 7
    return np.where(e == 0, (m / 8.0) * 2.0 ** -6, (1.0 + m / 8.0) * 2.0 ** (e.astype(np.float64) - 7))


def f32_to_e4m3_bits(x: np.ndarray) -> np.ndarray:
    """fp32 -> E4M3 code (uint8): round to nearest, ties to the even code, saturating at +-448."""
    x = np.ascontiguousarray(x, dtype=np.float32).astype(np.float64)
    mags = _e4m3_magnitudes()
    mids = (mags[:-1] + mags[1:]) / 2.0
    a = np.abs(x)
    idx = np.searchsorted(mids, a, side="left")               # midpoints strictly below |x|
    tie = (idx < mids.size) & (a == mids[np.minimum(idx, mids.size - 1)])
    idx = np.where(tie & (idx % 2 == 1), idx + 1, idx)        # exact tie: take the even code
    idx = np.minimum(idx, 126).astype(np.uint8)               # saturate to 448
    return (idx | (np.signbit(x).astype(np.uint8) << 7)).astype(np.uint8)


def make_fp8_case(M: int, N: int, K: int, seed: int, std: float = W_STD):
    """(A8 [M,K], W1_8 [N,K], W2_8 [N,K], scale_gate, scale_up): A ~ N(0,1) quantised directly;
    W ~ N(0, std) quantised as W / std (so the codes span the format) with dequantisation scale
    std folded into scale_gate = scale_up = std.  Weights in the [N,K] (nn.Linear) layout."""
    gen = lambda key, count: np.random.Generator(np.random.Philox(key=int(key))).standard_normal(
        count, dtype=np.float32)
    a8 = f32_to_e4m3_bits(gen(4 * seed + 2, M * K)).reshape(M, K)
    w1 = f32_to_e4m3_bits(gen(4 * seed + 0, N * K)).reshape(N, K)
    w2 = f32_to_e4m3_bits(gen(4 * seed + 1, N * K)).reshape(N, K)
    return a8, w1, w2, float(std), float(std)
