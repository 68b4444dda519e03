"""Thin ctypes binding over libswiglu_b200.so -- same names as include/swiglu_mlp.h.

Argument marshalling only: every step of the computation runs in the library's CUDA
kernels.  Tensors may be torch CUDA tensors (bf16, contiguous) or raw integer device
pointers together with explicit M, N, K.  There is no fallback of any kind: if the library
has not been built, loading raises; if there is no sm_100 device, the calls raise
SwigluError with the library's status code.
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libswiglu_b200.so")

SWIGLU_OK = 0
SWIGLU_ERR_NULL_POINTER = 1
SWIGLU_ERR_BAD_SHAPE = 2
SWIGLU_ERR_UNSUPPORTED = 3
SWIGLU_ERR_MISALIGNED = 4
SWIGLU_ERR_ALIASING = 5
SWIGLU_ERR_ARCH = 6
SWIGLU_ERR_WORKSPACE = 7
SWIGLU_ERR_CUDA = 8

EXPORTS = (
    "swiglu_mlp", "swiglu_mlp_unfused", "swiglu_mlp_ex", "swiglu_mlp_unfused_ex", "swiglu_silu_mul",
    "swiglu_glu_mlp", "swiglu_glu_mlp_unfused", "swiglu_glu_mlp_ex", "swiglu_act_mul",
    "swiglu_activation_name", "swiglu_glu_mlp_layout", "swiglu_mlp_host_batched",
    "swiglu_workspace_bytes", "swiglu_num_variants", "swiglu_variant_name",
    "swiglu_selected_variant", "swiglu_launches_per_call", "swiglu_validate",
    "swiglu_mlp_host", "swiglu_last_error", "swiglu_status_string", "swiglu_version",
    "swiglu_release", "swiglu_release_stream", "swiglu_reload_env", "swiglu_tensor_map_cache_stats",
    "swiglu_set_clock_probe", "swiglu_packed_weight_bytes", "swiglu_pack_weights",
    "swiglu_mlp_packed", "swiglu_glu_mlp_packed", "swiglu_launch_floor_probe",
    "swiglu_mlp_fp8", "swiglu_mlp_fp8_ex", "swiglu_mlp_unfused_static",
)


class SwigluError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{status_string(status)} ({status}): {message}")
        self.status = status


_lib = None


def load():
    """Load the C-ABI library.  Raises (loudly) if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2607_02521_b200.build` "
            "(or __graft_entry__.build()); there is no CPU or PyTorch fallback")
    lib = ctypes.CDLL(LIB_PATH)
    p, i64, sz, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_size_t, ctypes.c_int
    for name in ("swiglu_mlp", "swiglu_mlp_unfused", "swiglu_mlp_unfused_static"):
        f = getattr(lib, name)
        f.argtypes, f.restype = [p, p, p, p, i64, i64, i64, p], ci
    for name in ("swiglu_mlp_ex", "swiglu_mlp_unfused_ex"):
        f = getattr(lib, name)
        f.argtypes, f.restype = [p, p, p, p, i64, i64, i64, p, sz, ci, p], ci
    lib.swiglu_workspace_bytes.argtypes, lib.swiglu_workspace_bytes.restype = [i64, i64, i64, ci, ci], sz
    lib.swiglu_num_variants.argtypes, lib.swiglu_num_variants.restype = [ci], ci
    lib.swiglu_variant_name.argtypes, lib.swiglu_variant_name.restype = [ci, ci], ctypes.c_char_p
    lib.swiglu_selected_variant.argtypes, lib.swiglu_selected_variant.restype = [i64, i64, i64, ci], ci
    lib.swiglu_launches_per_call.argtypes, lib.swiglu_launches_per_call.restype = [i64, i64, i64, ci, ci], ci
    lib.swiglu_validate.argtypes, lib.swiglu_validate.restype = [p, p, p, p, i64, i64, i64], ci
    lib.swiglu_mlp_host.argtypes, lib.swiglu_mlp_host.restype = [p, p, p, p, i64, i64, i64, ci, p], ci
    lib.swiglu_silu_mul.argtypes, lib.swiglu_silu_mul.restype = [p, p, p, i64, p], ci
    lib.swiglu_act_mul.argtypes, lib.swiglu_act_mul.restype = [p, p, p, i64, ci, p], ci
    for name in ("swiglu_glu_mlp", "swiglu_glu_mlp_unfused"):
        f = getattr(lib, name)
        f.argtypes, f.restype = [p, p, p, p, i64, i64, i64, ci, p], ci
    lib.swiglu_glu_mlp_ex.argtypes = [p, p, p, p, i64, i64, i64, ci, ci, p]
    lib.swiglu_glu_mlp_ex.restype = ci
    lib.swiglu_activation_name.argtypes, lib.swiglu_activation_name.restype = [ci], ctypes.c_char_p
    lib.swiglu_glu_mlp_layout.argtypes = [p, p, p, p, i64, i64, i64, ci, ci, ci, ci, p]
    lib.swiglu_glu_mlp_layout.restype = ci
    lib.swiglu_mlp_host_batched.argtypes = [p, p, p, ci, p, p, i64, i64, ci, p]
    lib.swiglu_mlp_host_batched.restype = ci
    lib.swiglu_release.argtypes, lib.swiglu_release.restype = [], ci
    lib.swiglu_release_stream.argtypes, lib.swiglu_release_stream.restype = [p], ci
    lib.swiglu_reload_env.argtypes, lib.swiglu_reload_env.restype = [], None
    u64p = ctypes.POINTER(ctypes.c_uint64)
    lib.swiglu_tensor_map_cache_stats.argtypes, lib.swiglu_tensor_map_cache_stats.restype = [u64p, u64p], ci
    lib.swiglu_set_clock_probe.argtypes, lib.swiglu_set_clock_probe.restype = [p], None
    lib.swiglu_packed_weight_bytes.argtypes, lib.swiglu_packed_weight_bytes.restype = [i64, i64], sz
    lib.swiglu_pack_weights.argtypes, lib.swiglu_pack_weights.restype = [p, p, p, i64, i64, ci, p], ci
    lib.swiglu_mlp_packed.argtypes, lib.swiglu_mlp_packed.restype = [p, p, p, i64, i64, i64, p], ci
    lib.swiglu_glu_mlp_packed.argtypes = [p, p, p, i64, i64, i64, ci, ci, p]
    lib.swiglu_glu_mlp_packed.restype = ci
    cf = ctypes.c_float
    lib.swiglu_mlp_fp8.argtypes, lib.swiglu_mlp_fp8.restype = [p, p, p, p, i64, i64, i64, cf, cf, p], ci
    lib.swiglu_mlp_fp8_ex.argtypes = [p, p, p, p, i64, i64, i64, cf, cf, ci, p]
    lib.swiglu_mlp_fp8_ex.restype = ci
    lib.swiglu_launch_floor_probe.argtypes = [p, p, p, p, i64, i64, i64, p]
    lib.swiglu_launch_floor_probe.restype = ci
    lib.swiglu_last_error.argtypes, lib.swiglu_last_error.restype = [], ctypes.c_char_p
    lib.swiglu_status_string.argtypes, lib.swiglu_status_string.restype = [ci], ctypes.c_char_p
    lib.swiglu_version.argtypes, lib.swiglu_version.restype = [], ctypes.c_char_p
    _lib = lib
    return lib


# ------------------------------------------------------------------ marshalling helpers
def _ptr(x):
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):      # torch.Tensor
        return int(x.data_ptr())
    if hasattr(x, "ctypes"):        # numpy array (host buffers of swiglu_mlp_host)
        return int(x.ctypes.data)
    raise TypeError(f"cannot take a pointer from {type(x)}")


def _stream(stream):
    if stream is None:
        try:
            import torch
            if torch.cuda.is_available():
                return int(torch.cuda.current_stream().cuda_stream)
        except ImportError:
            pass
        return None
    if isinstance(stream, int):
        return stream or None
    return int(stream.cuda_stream)


def _dims(A, W1, W2, Y, M, N, K):
    if M is not None and N is not None and K is not None:
        return int(M), int(N), int(K)
    for t, name in ((A, "A"), (W1, "W1"), (W2, "W2"), (Y, "Y")):
        if not hasattr(t, "shape") or len(t.shape) != 2:
            raise TypeError(f"{name}: need a 2-D tensor, or pass M, N, K with raw pointers")
        if hasattr(t, "is_contiguous") and not t.is_contiguous():
            raise ValueError(f"{name} must be contiguous (dense row-major, no strides)")
        if hasattr(t, "element_size") and t.element_size() != 2:
            raise TypeError(f"{name} must hold 2-byte bf16 elements")
    m, k = A.shape
    k2, n = W1.shape
    if k2 != k or tuple(W2.shape) != (k, n) or tuple(Y.shape) != (m, n):
        raise ValueError(f"shape mismatch: A{tuple(A.shape)} W1{tuple(W1.shape)} "
                         f"W2{tuple(W2.shape)} Y{tuple(Y.shape)}")
    return int(m), int(n), int(k)


def _check(status: int):
    if status != SWIGLU_OK:
        raise SwigluError(status, last_error())


# ------------------------------------------------------------------ the ABI, name for name
def swiglu_mlp(A, W1, W2, Y, M=None, N=None, K=None, stream=None) -> None:
    """Fused Y = bf16(SiLU(A.W1) * (A.W2)); asynchronous on `stream`."""
    m, n, k = _dims(A, W1, W2, Y, M, N, K)
    _check(load().swiglu_mlp(_ptr(A), _ptr(W1), _ptr(W2), _ptr(Y), m, n, k, _stream(stream)))


def swiglu_mlp_unfused(A, W1, W2, Y, M=None, N=None, K=None, stream=None) -> None:
    """Unfused comparison path: two GEMMs writing bf16 Gate/Up, then SiLU-multiply."""
    m, n, k = _dims(A, W1, W2, Y, M, N, K)
    _check(load().swiglu_mlp_unfused(_ptr(A), _ptr(W1), _ptr(W2), _ptr(Y), m, n, k,
                                     _stream(stream)))


STATIC_SCRATCH_BYTES = 32 << 20   # SWIGLU_STATIC_SCRATCH_BYTES


def swiglu_mlp_unfused_static(A, W1, W2, Y, M=None, N=None, K=None, stream=None) -> None:
    """swiglu_mlp_unfused with its Gate/Up scratch in the library's static device array: no
    allocation; sizes beyond STATIC_SCRATCH_BYTES are rejected; overlapping calls race."""
    m, n, k = _dims(A, W1, W2, Y, M, N, K)
    _check(load().swiglu_mlp_unfused_static(_ptr(A), _ptr(W1), _ptr(W2), _ptr(Y), m, n, k,
                                            _stream(stream)))


def swiglu_mlp_ex(A, W1, W2, Y, M=None, N=None, K=None, workspace=None, workspace_bytes=0,
                  variant=-1, stream=None) -> None:
    m, n, k = _dims(A, W1, W2, Y, M, N, K)
    _check(load().swiglu_mlp_ex(_ptr(A), _ptr(W1), _ptr(W2), _ptr(Y), m, n, k, _ptr(workspace),
                                int(workspace_bytes), int(variant), _stream(stream)))


def swiglu_mlp_unfused_ex(A, W1, W2, Y, M=None, N=None, K=None, workspace=None,
                          workspace_bytes=0, variant=-1, stream=None) -> None:
    m, n, k = _dims(A, W1, W2, Y, M, N, K)
    _check(load().swiglu_mlp_unfused_ex(_ptr(A), _ptr(W1), _ptr(W2), _ptr(Y), m, n, k,
                                        _ptr(workspace), int(workspace_bytes), int(variant),
                                        _stream(stream)))


ACTIVATIONS = {"silu": 0, "gelu": 1, "gelu_tanh": 2, "relu": 3}   # swiglu_activation ids


def _act(activation) -> int:
    return int(ACTIVATIONS.get(activation, activation))


def swiglu_glu_mlp(A, W1, W2, Y, activation, M=None, N=None, K=None, stream=None) -> None:
    """Y = bf16(act(A.W1) * (A.W2)), act = "silu" | "gelu" | "gelu_tanh" | "relu" (or its id)."""
    m, n, k = _dims(A, W1, W2, Y, M, N, K)
    _check(load().swiglu_glu_mlp(_ptr(A), _ptr(W1), _ptr(W2), _ptr(Y), m, n, k, _act(activation),
                                 _stream(stream)))


def swiglu_glu_mlp_unfused(A, W1, W2, Y, activation, M=None, N=None, K=None, stream=None) -> None:
    m, n, k = _dims(A, W1, W2, Y, M, N, K)
    _check(load().swiglu_glu_mlp_unfused(_ptr(A), _ptr(W1), _ptr(W2), _ptr(Y), m, n, k,
                                         _act(activation), _stream(stream)))


def swiglu_glu_mlp_ex(A, W1, W2, Y, activation, variant=-1, M=None, N=None, K=None,
                      stream=None) -> None:
    m, n, k = _dims(A, W1, W2, Y, M, N, K)
    _check(load().swiglu_glu_mlp_ex(_ptr(A), _ptr(W1), _ptr(W2), _ptr(Y), m, n, k,
                                    _act(activation), int(variant), _stream(stream)))


WEIGHTS_KN, WEIGHTS_NK = 0, 1   # swiglu_weight_layout


def swiglu_glu_mlp_layout(A, W1, W2, Y, activation="silu", weight_layout=WEIGHTS_NK, unfused=False,
                          variant=-1, M=None, N=None, K=None, stream=None) -> None:
    """As swiglu_glu_mlp with W1, W2 given as [N, K] row-major (weight_layout=WEIGHTS_NK, the
    nn.Linear layout) or [K, N] (WEIGHTS_KN)."""
    if M is None:
        M, K = int(A.shape[0]), int(A.shape[1])
        N = int(Y.shape[1])
    _check(load().swiglu_glu_mlp_layout(_ptr(A), _ptr(W1), _ptr(W2), _ptr(Y), int(M), int(N), int(K),
                                        _act(activation), int(weight_layout), int(bool(unfused)),
                                        int(variant), _stream(stream)))


def swiglu_act_mul(G, U, Y, activation, elems=None, stream=None) -> None:
    if elems is None:
        elems = int(G.numel())
    _check(load().swiglu_act_mul(_ptr(G), _ptr(U), _ptr(Y), int(elems), _act(activation),
                                 _stream(stream)))


def swiglu_activation_name(activation: int):
    r = load().swiglu_activation_name(int(activation))
    return r.decode() if r else None


def swiglu_silu_mul(G, U, Y, elems=None, stream=None) -> None:
    """Elementwise stage alone: Y = bf16(SiLU(G) * U) over `elems` bf16 values (device)."""
    if elems is None:
        elems = int(G.numel())
    _check(load().swiglu_silu_mul(_ptr(G), _ptr(U), _ptr(Y), int(elems), _stream(stream)))


def swiglu_mlp_host(A_host, W1_host, W2_host, Y_host, M, N, K, unfused=False, stream=None) -> None:
    """Host-buffer form: H2D copies, the kernel(s), D2H copy and a stream sync, all inside."""
    _check(load().swiglu_mlp_host(_ptr(A_host), _ptr(W1_host), _ptr(W2_host), _ptr(Y_host),
                                  int(M), int(N), int(K), int(bool(unfused)), _stream(stream)))


def swiglu_mlp_host_batched(A_hosts, Y_hosts, Ms, W1_host, W2_host, N, K, unfused=False,
                            stream=None) -> None:
    """One set of host weights, several host activation batches: weights cross PCIe once, in
    column chunks pipelined with the kernels and the downloads (see the header)."""
    n = len(Ms)
    a = (ctypes.c_void_p * n)(*[_ptr(x) for x in A_hosts])
    y = (ctypes.c_void_p * n)(*[_ptr(x) for x in Y_hosts])
    m = (ctypes.c_int64 * n)(*[int(v) for v in Ms])
    _check(load().swiglu_mlp_host_batched(a, y, m, n, _ptr(W1_host), _ptr(W2_host), int(N), int(K),
                                          int(bool(unfused)), _stream(stream)))


def swiglu_validate(A, W1, W2, Y, M, N, K) -> int:
    """Returns the status code (no exception): the argument checks, without any CUDA call."""
    return int(load().swiglu_validate(_ptr(A), _ptr(W1), _ptr(W2), _ptr(Y), int(M), int(N), int(K)))


def swiglu_workspace_bytes(M, N, K, unfused=False, variant=-1) -> int:
    return int(load().swiglu_workspace_bytes(int(M), int(N), int(K), int(bool(unfused)), int(variant)))


def swiglu_num_variants(unfused=False) -> int:
    return int(load().swiglu_num_variants(int(bool(unfused))))


def swiglu_variant_name(variant, unfused=False):
    s = load().swiglu_variant_name(int(bool(unfused)), int(variant))
    return None if s is None else s.decode()


def swiglu_selected_variant(M, N, K, unfused=False) -> int:
    return int(load().swiglu_selected_variant(int(M), int(N), int(K), int(bool(unfused))))


def swiglu_launches_per_call(M, N, K, unfused=False, variant=-1) -> int:
    return int(load().swiglu_launches_per_call(int(M), int(N), int(K), int(bool(unfused)), int(variant)))


def swiglu_release() -> None:
    """Synchronise the device and free every library-owned buffer, copy stream and event."""
    _check(load().swiglu_release())


def swiglu_release_stream(stream=None) -> None:
    """Stream-ordered free of the library's buffers for `stream` (no synchronisation)."""
    _check(load().swiglu_release_stream(_stream(stream)))


def swiglu_reload_env() -> None:
    """Re-read the SWIGLU_* experiment overrides from the environment (sweeps / tests)."""
    load().swiglu_reload_env()


def swiglu_tensor_map_cache_stats():
    """(hits, misses, slots) of the calling thread's tensor-map cache."""
    h, m = ctypes.c_uint64(0), ctypes.c_uint64(0)
    slots = load().swiglu_tensor_map_cache_stats(ctypes.byref(h), ctypes.byref(m))
    return int(h.value), int(m.value), int(slots)


def swiglu_packed_weight_bytes(N, K) -> int:
    return int(load().swiglu_packed_weight_bytes(int(N), int(K)))


def swiglu_pack_weights(W1, W2, Wp, N, K, weight_layout=WEIGHTS_KN, stream=None) -> None:
    """One-time prepack of (W1, W2) into the tile-interleaved W_fused buffer Wp (device)."""
    _check(load().swiglu_pack_weights(_ptr(W1), _ptr(W2), _ptr(Wp), int(N), int(K),
                                      int(weight_layout), _stream(stream)))


def swiglu_mlp_packed(A, Wp, Y, M=None, N=None, K=None, stream=None) -> None:
    """Fused Y = bf16(SiLU(A.W1) * (A.W2)) from prepacked weights (see the header's contract)."""
    if M is None:
        M, K = int(A.shape[0]), int(A.shape[1])
        N = int(Y.shape[1])
    _check(load().swiglu_mlp_packed(_ptr(A), _ptr(Wp), _ptr(Y), int(M), int(N), int(K),
                                    _stream(stream)))


def swiglu_glu_mlp_packed(A, Wp, Y, activation="silu", variant=-1, M=None, N=None, K=None,
                          stream=None) -> None:
    if M is None:
        M, K = int(A.shape[0]), int(A.shape[1])
        N = int(Y.shape[1])
    _check(load().swiglu_glu_mlp_packed(_ptr(A), _ptr(Wp), _ptr(Y), int(M), int(N), int(K),
                                        _act(activation), int(variant), _stream(stream)))


def swiglu_mlp_fp8(A8, W1_8, W2_8, Y, scale_gate=1.0, scale_up=1.0, variant=-1, M=None, N=None,
                   K=None, stream=None) -> None:
    """FP8 (E4M3) operands: Y = bf16(SiLU(scale_gate * A8.W1_8^T) * (scale_up * A8.W2_8^T));
    A8 [M,K], W1_8 / W2_8 [N,K] one byte per element, Y [M,N] bf16."""
    if M is None:
        M, K = int(A8.shape[0]), int(A8.shape[1])
        N = int(Y.shape[1])
    _check(load().swiglu_mlp_fp8_ex(_ptr(A8), _ptr(W1_8), _ptr(W2_8), _ptr(Y), int(M), int(N),
                                    int(K), float(scale_gate), float(scale_up), int(variant),
                                    _stream(stream)))


def swiglu_launch_floor_probe(A, W1, W2, Y, M=None, N=None, K=None, stream=None) -> None:
    """Measurement aid: the decode kernel's launch with an empty body (see the header)."""
    m, n, k = _dims(A, W1, W2, Y, M, N, K)
    _check(load().swiglu_launch_floor_probe(_ptr(A), _ptr(W1), _ptr(W2), _ptr(Y), m, n, k,
                                            _stream(stream)))


def swiglu_set_clock_probe(buf) -> None:
    """Register (or, with None, clear) a device buffer of two uint64 {SM cycles, ns} that CTA 0
    of every GEMM-class launch fills in; see the header."""
    load().swiglu_set_clock_probe(_ptr(buf))


def last_error() -> str:
    return load().swiglu_last_error().decode()


swiglu_last_error = last_error


def status_string(status: int) -> str:
    return load().swiglu_status_string(int(status)).decode()


swiglu_status_string = status_string


def swiglu_version() -> str:
    return load().swiglu_version().decode()
