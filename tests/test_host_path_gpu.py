"""Host path of the C ABI on a real device: tensor-map cache,
library-owned buffers (stream-ordered growth, release, stream handle reuse), call overhead,
and the host-buffer pipeline's scratch layout."""
import time

import numpy as np
import pytest
import torch

import oracle
from paper_2607_02521_b200 import binding as B
from paper_2607_02521_b200 import check, inputs

pytestmark = pytest.mark.gpu


def dev(bits):
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).cuda().view(torch.bfloat16)


def host(t):
    return t.view(torch.int16).cpu().numpy().view(np.uint16)


def test_tensor_maps_are_encoded_once_per_distinct_tensor():
    M, N, K = 16, 392, 328
    A, W1, W2 = inputs.make_case(M, N, K, seed=11, std=0.05)
    dA, dW1, dW2 = dev(A), dev(W1), dev(W2)
    dY = torch.empty((M, N), dtype=torch.bfloat16, device="cuda")
    B.swiglu_mlp(dA, dW1, dW2, dY)
    h0, m0, _ = B.swiglu_tensor_map_cache_stats()
    for _ in range(50):
        B.swiglu_mlp(dA, dW1, dW2, dY)
    h1, m1, _ = B.swiglu_tensor_map_cache_stats()
    torch.cuda.synchronize()
    assert m1 == m0, "repeat calls on the same tensors must not re-encode"
    assert h1 - h0 >= 50 * 3
    y_ref, _ = oracle.swiglu_oracle(A, W1, W2)
    assert check.compare(host(dY), y_ref).mismatches == 0
    # a different tensor at another address misses once, then hits
    dA2 = dA.clone()
    B.swiglu_mlp(dA2, dW1, dW2, dY)
    h2, m2, _ = B.swiglu_tensor_map_cache_stats()
    # (one encode for the new tensor; the table is 4-way set associative with LRU replacement, so
    # the few live maps of these calls cannot evict each other wherever the allocator put them)
    assert m2 == m1 + 1
    for _ in range(20):
        B.swiglu_mlp(dA2, dW1, dW2, dY)
        B.swiglu_mlp(dA, dW1, dW2, dY)
    h3, m3, _ = B.swiglu_tensor_map_cache_stats()
    assert m3 == m2 and h3 - h2 >= 40 * 3, "both activation buffers' maps stay cached"
    torch.cuda.synchronize()


def test_host_call_overhead_of_tiny_shapes():
    """Eager (non-graph) calls of a tiny shape on the NULL stream: the host side (validation,
    dispatch, cached tensor maps, cudaLaunchKernelEx) must sustain well over 50k calls/s."""
    M, N, K = 8, 128, 64
    A, W1, W2 = inputs.make_case(M, N, K, seed=12)
    dA, dW1, dW2 = dev(A), dev(W1), dev(W2)
    dY = torch.empty((M, N), dtype=torch.bfloat16, device="cuda")
    lib = B.load()
    args = (dA.data_ptr(), dW1.data_ptr(), dW2.data_ptr(), dY.data_ptr(), M, N, K, None)
    for _ in range(200):
        assert lib.swiglu_mlp(*args) == 0
    torch.cuda.synchronize()
    n = 5000
    t_enqueue = float("inf")
    for _ in range(3):                       # best of three: robust to a hiccup of the host
        t0 = time.perf_counter()
        for _ in range(n):
            lib.swiglu_mlp(*args)
        t_enqueue = min(t_enqueue, time.perf_counter() - t0)
        torch.cuda.synchronize()
    rate = n / t_enqueue
    print(f"host enqueue rate: {rate:,.0f} calls/s ({1e6 * t_enqueue / n:.2f} us per call)")
    assert rate > 50_000
    y_ref, _ = oracle.swiglu_oracle(A, W1, W2)
    assert check.compare(host(dY), y_ref).mismatches == 0


def test_stream_create_destroy_reuse_and_release():
    """Library-owned per-stream buffers across stream lifetimes: grow on a stream, release it,
    destroy it, create new streams (handles get reused), call again; then swiglu_release()."""
    K, N = 200, 1032
    A_all, W1, W2 = inputs.make_case(300, N, K, seed=13, std=0.05)
    y_ref, _ = oracle.swiglu_oracle(A_all, W1, W2)
    dW1, dW2 = dev(W1), dev(W2)
    for rnd in range(6):
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            for M in (5, 300, 40):                  # grow, then a smaller call on the same buffer
                dA = dev(A_all[:M])
                dY = torch.full((M, N), float("nan"), dtype=torch.bfloat16, device="cuda")
                B.swiglu_mlp_unfused(dA, dW1, dW2, dY, stream=st)
                st.synchronize()
                assert check.compare(host(dY), y_ref[:M]).mismatches == 0, (rnd, M)
            if rnd % 2 == 0:
                B.swiglu_release_stream(st)
        del st
    B.swiglu_release()
    # the library is still usable after a full release
    dA = dev(A_all[:64])
    dY = torch.full((64, N), float("nan"), dtype=torch.bfloat16, device="cuda")
    B.swiglu_mlp_unfused(dA, dW1, dW2, dY)
    Yh = np.zeros((64, N), dtype=np.uint16)
    B.swiglu_mlp_host(A_all[:64], W1, W2, Yh, 64, N, K)
    torch.cuda.synchronize()
    assert check.compare(host(dY), y_ref[:64]).mismatches == 0
    assert check.compare(Yh, y_ref[:64]).mismatches == 0


def test_library_workspace_is_refused_under_capture():
    """A captured graph would keep a pointer that the next growth frees: the 8-argument unfused
    form refuses a capturing stream; the _ex form with a caller workspace captures fine."""
    M, N, K = 16, 392, 328
    A, W1, W2 = inputs.make_case(M, N, K, seed=14, std=0.05)
    dA, dW1, dW2 = dev(A), dev(W1), dev(W2)
    dY = torch.zeros((M, N), dtype=torch.bfloat16, device="cuda")
    B.swiglu_mlp_unfused(dA, dW1, dW2, dY)           # buffer exists and is large enough
    torch.cuda.synchronize()
    need = B.swiglu_workspace_bytes(M, N, K, unfused=True)
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        with pytest.raises(B.SwigluError) as e:
            B.swiglu_mlp_unfused(dA, dW1, dW2, dY)
        assert e.value.status == B.SWIGLU_ERR_WORKSPACE
        B.swiglu_mlp_unfused_ex(dA, dW1, dW2, dY, workspace=ws, workspace_bytes=need)
    dY.zero_()
    g.replay()
    torch.cuda.synchronize()
    y_ref, _ = oracle.swiglu_oracle(A, W1, W2)
    assert check.compare(host(dY), y_ref).mismatches == 0


@pytest.mark.parametrize("N", [8, 264])
@pytest.mark.parametrize("unfused", [False, True])
def test_host_batched_many_small_batches_narrow_n(N, unfused):
    """with N < 512 and N % 128 != 0 the per-batch 256-byte padding of the Y scratch
    used to add up past the allocation.  Many batches, narrow N, every output checked; the
    device scratch sits in the library's own buffer, so an overrun would corrupt a neighbour
    batch's rows (all rows are compared) or fault."""
    K = 72
    Ms = [1] * 40 + [3, 0, 7, 2] * 6
    A_all, W1, W2 = inputs.make_case(sum(Ms), N, K, seed=900 + N, std=0.05)
    y_ref, _ = oracle.swiglu_oracle(A_all, W1, W2)
    offs = np.cumsum([0] + Ms)
    mk = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.int16)).pin_memory()
    hA = [mk(A_all[offs[i]:offs[i + 1]]) if Ms[i] else None for i in range(len(Ms))]
    hY = [mk(np.full((Ms[i], N), 0x7FC0, dtype=np.uint16)) if Ms[i] else None for i in range(len(Ms))]
    B.swiglu_mlp_host_batched(hA, hY, Ms, mk(W1), mk(W2), N, K, unfused=unfused)
    for i, M in enumerate(Ms):
        if M:
            rep = check.compare(hY[i].numpy().view(np.uint16), y_ref[offs[i]:offs[i + 1]])
            assert rep.mismatches == 0, (i, M, rep)
