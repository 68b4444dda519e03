"""ctypes loader for ``swiglu_oracle.c``.  TEST INFRASTRUCTURE ONLY (see ``__init__``).

No arithmetic of the method happens in this file: it checks shapes/dtypes, hands the
pointers to the C functions and returns their fp64 output.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "swiglu_oracle.c")
_LIB = os.path.join(_HERE, "libswiglu_oracle.so")
_lock = threading.Lock()
_lib = None

# -O2, OpenMP; no -ffast-math, and no FMA contraction, so every a*w product and every
# += rounds exactly as written in the C source.
_CFLAGS = ["-O2", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
           "-std=c11", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (idempotent).  Returns the path of the shared object."""
    with _lock:
        stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
        if force or stale:
            tmp = _LIB + ".tmp.%d" % os.getpid()
            subprocess.run(["gcc", *_CFLAGS, "-o", tmp, _SRC, "-lm"], check=True)
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        path = build()
        lib = ctypes.CDLL(path)
        i64, p = ctypes.c_int64, ctypes.c_void_p
        lib.swiglu_oracle.argtypes = [p, p, p, p, i64, i64, i64, ctypes.c_int]
        lib.swiglu_oracle.restype = ctypes.c_int
        lib.swiglu_oracle_rows.argtypes = [p, p, p, p, p, i64, i64, i64, i64, ctypes.c_int]
        lib.swiglu_oracle_rows.restype = ctypes.c_int
        lib.swiglu_oracle_act.argtypes = [p, p, p, p, i64, i64, i64, ctypes.c_int, ctypes.c_int]
        lib.swiglu_oracle_act.restype = ctypes.c_int
        lib.swiglu_oracle_rows_act.argtypes = [p, p, p, p, p, i64, i64, i64, i64, ctypes.c_int,
                                               ctypes.c_int]
        lib.swiglu_oracle_rows_act.restype = ctypes.c_int
        lib.swiglu_oracle_activation.argtypes = [ctypes.c_int, ctypes.c_double]
        lib.swiglu_oracle_activation.restype = ctypes.c_double
        lib.swiglu_oracle_silu.argtypes = [ctypes.c_double]
        lib.swiglu_oracle_silu.restype = ctypes.c_double
        lib.swiglu_oracle_e4m3_to_f64.argtypes = [ctypes.c_uint8]
        lib.swiglu_oracle_e4m3_to_f64.restype = ctypes.c_double
        lib.swiglu_oracle_fp8_rows.argtypes = [p, p, p, p, p, i64, i64, i64, i64, ctypes.c_double,
                                               ctypes.c_double, ctypes.c_int]
        lib.swiglu_oracle_fp8_rows.restype = ctypes.c_int
        lib.swiglu_oracle_pack_rows.argtypes, lib.swiglu_oracle_pack_rows.restype = [i64], i64
        lib.swiglu_oracle_pack.argtypes = [p, p, p, i64, i64]
        lib.swiglu_oracle_pack.restype = ctypes.c_int
        lib.swiglu_oracle_max_threads.argtypes = []
        lib.swiglu_oracle_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _bits(x, shape, name):
    a = np.ascontiguousarray(x)
    if a.dtype != np.uint16:
        raise TypeError(f"{name}: expected bf16 bit patterns as uint16, got {a.dtype}")
    if a.shape != shape:
        raise ValueError(f"{name}: expected shape {shape}, got {a.shape}")
    return a


def _ptr(a):
    return ctypes.c_void_p(a.ctypes.data)


def max_threads() -> int:
    return int(_load().swiglu_oracle_max_threads())


def silu(x: float) -> float:
    """The oracle's own fp64 SiLU (exposed so the pins can probe it directly)."""
    return float(_load().swiglu_oracle_silu(float(x)))


ACTIVATIONS = {"silu": 0, "gelu": 1, "gelu_tanh": 2, "relu": 3}


def activation(act, x: float) -> float:
    """The oracle's own fp64 gate activation (act: name or id), for the pins."""
    return float(_load().swiglu_oracle_activation(int(ACTIVATIONS.get(act, act)), float(x)))


def swiglu_oracle(A_bits, W1_bits, W2_bits, nthreads: int = 0, act=0):
    """y_ref[M,N] in fp64 from bf16 bit patterns A[M,K], W1[K,N], W2[K,N] (uint16);
    act = 0/"silu" (the paper's Eq. 3), "gelu", "gelu_tanh", "relu" (GeGLU / ReGLU).

    Returns (y_ref, threads_used)."""
    A_bits = np.ascontiguousarray(A_bits)
    W1_bits = np.ascontiguousarray(W1_bits)
    if A_bits.ndim != 2 or W1_bits.ndim != 2:
        raise ValueError("A and W1 must be 2-D")
    M, K = A_bits.shape
    K2, N = W1_bits.shape
    if K2 != K:
        raise ValueError(f"A is [{M},{K}] but W1 is [{K2},{N}]")
    A = _bits(A_bits, (M, K), "A")
    W1 = _bits(W1_bits, (K, N), "W1")
    W2 = _bits(W2_bits, (K, N), "W2")
    Y = np.empty((M, N), dtype=np.float64)
    used = _load().swiglu_oracle_act(_ptr(A), _ptr(W1), _ptr(W2), _ptr(Y), M, N, K,
                                     int(ACTIVATIONS.get(act, act)), int(nthreads))
    if used < 0:
        raise RuntimeError("swiglu_oracle rejected its arguments")
    return Y, int(used)


def swiglu_oracle_rows(A_bits, W1_bits, W2_bits, rows, nthreads: int = 0, act=0):
    """Rows ``rows`` of y_ref only (full N columns each): [len(rows), N] fp64."""
    A_bits = np.ascontiguousarray(A_bits)
    W1_bits = np.ascontiguousarray(W1_bits)
    M, K = A_bits.shape
    K2, N = W1_bits.shape
    if K2 != K:
        raise ValueError(f"A is [{M},{K}] but W1 is [{K2},{N}]")
    A = _bits(A_bits, (M, K), "A")
    W1 = _bits(W1_bits, (K, N), "W1")
    W2 = _bits(W2_bits, (K, N), "W2")
    r = np.ascontiguousarray(np.asarray(rows, dtype=np.int64))
    Y = np.empty((r.shape[0], N), dtype=np.float64)
    used = _load().swiglu_oracle_rows_act(_ptr(A), _ptr(W1), _ptr(W2), _ptr(Y), _ptr(r),
                                          r.shape[0], M, N, K, int(ACTIVATIONS.get(act, act)),
                                          int(nthreads))
    if used < 0:
        raise RuntimeError("swiglu_oracle_rows rejected its arguments")
    return Y, int(used)


def pack_rows(K: int) -> int:
    """Rows per slab of the W_fused buffer (K plus its padding rows)."""
    return int(_load().swiglu_oracle_pack_rows(int(K)))


def pack_weights(W1_bits, W2_bits):
    """The one-time W_fused interleave (swiglu_oracle.c
    swiglu_oracle_pack): uint16 [ceil(N/128), 4, Kp, 64] from W1, W2 [K, N] bit patterns, Kp = K
    plus 8 or 16 zero padding rows per slab (pack_rows)."""
    W1_bits = np.ascontiguousarray(W1_bits)
    K, N = W1_bits.shape
    W1 = _bits(W1_bits, (K, N), "W1")
    W2 = _bits(W2_bits, (K, N), "W2")
    Wp = np.empty(((N + 127) // 128, 4, pack_rows(K), 64), dtype=np.uint16)
    if _load().swiglu_oracle_pack(_ptr(W1), _ptr(W2), _ptr(Wp), N, K) != 0:
        raise RuntimeError("swiglu_oracle_pack rejected its arguments")
    return Wp


def e4m3_to_f64(code: int) -> float:
    """The oracle's own decode of one OCP FP8 E4M3 code (for the pins)."""
    return float(_load().swiglu_oracle_e4m3_to_f64(int(code) & 0xFF))


def swiglu_oracle_fp8(A8, W1_8, W2_8, scale_gate=1.0, scale_up=1.0, rows=None, nthreads: int = 0):
    """FP8 (E4M3) operands: y_ref = SiLU(scale_gate * A8.W1_8^T) * (scale_up * A8.W2_8^T) in fp64.
    A8 [M,K], W1_8 / W2_8 [N,K] (K contiguous), all uint8 codes.  rows: optional row subset.
    Returns (y_ref [len(rows) or M, N], threads_used)."""
    A = np.ascontiguousarray(A8)
    W1 = np.ascontiguousarray(W1_8)
    W2 = np.ascontiguousarray(W2_8)
    if A.dtype != np.uint8 or W1.dtype != np.uint8 or W2.dtype != np.uint8:
        raise TypeError("FP8 operands are passed as uint8 codes")
    M, K = A.shape
    N, K2 = W1.shape
    if K2 != K or W2.shape != (N, K):
        raise ValueError(f"A is [{M},{K}] but W1 is {W1.shape}, W2 is {W2.shape} (need [N,K])")
    r = None if rows is None else np.ascontiguousarray(np.asarray(rows, dtype=np.int64))
    count = M if r is None else r.shape[0]
    Y = np.empty((count, N), dtype=np.float64)
    used = _load().swiglu_oracle_fp8_rows(_ptr(A), _ptr(W1), _ptr(W2), _ptr(Y),
                                          None if r is None else _ptr(r), count, M, N, K,
                                          float(scale_gate), float(scale_up), int(nthreads))
    if used < 0:
        raise RuntimeError("swiglu_oracle_fp8 rejected its arguments")
    return Y, int(used)
