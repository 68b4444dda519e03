"""swiglu_mlp_unfused_static: the no-allocation entry point (include/swiglu_mlp.h).  Its Gate / Up
scratch is one file-scope `static __device__` array inside the library (32 MiB), so a caller that
cannot allocate device memory (CUDA-graph capture, tight serving loops) can still run the
unfused path.  Collected LAST on purpose (the suite runs with `pytest -x`).

The GPU test compares the new entry point with the existing path (`swiglu_mlp_unfused`: same
kernels, library-owned workspace) on two calls in a row that share the static array, within the
bound the other parity tests use, |y - y_ref| <= 2e-3 + 1.6e-2 |y_ref|, and against the oracle.
"""
import numpy as np
import pytest

from paper_2607_02521_b200 import binding as B
from paper_2607_02521_b200 import build as libbuild

ATOL, RTOL = 2e-3, 1.6e-2
# fake aligned pointers 64 GiB apart (never dereferenced: every check below fails or returns first)
A_, W1_, W2_, Y_ = 0x1000000000, 0x2000000000, 0x3000000000, 0x4000000000


def test_sizes_beyond_the_static_scratch_are_rejected_before_any_cuda_call():
    """Host-only: the size check precedes every CUDA call, so it answers on a box without a GPU."""
    libbuild.build()
    B.load()
    limit = B.STATIC_SCRATCH_BYTES
    assert limit == 32 << 20
    # the largest M that fits at N = 29568, and one row more
    N, K = 29568, 8192
    m_fit = limit // (2 * N * 2)
    assert B.swiglu_workspace_bytes(m_fit, N, K, unfused=True) <= limit
    assert B.swiglu_workspace_bytes(m_fit + 1, N, K, unfused=True) > limit
    with pytest.raises(B.SwigluError) as e:
        B.swiglu_mlp_unfused_static(A_, W1_, W2_, Y_, M=m_fit + 1, N=N, K=K, stream=0)
    assert e.value.status == B.SWIGLU_ERR_WORKSPACE
    assert "static scratch" in str(e.value)
    # the ordinary argument checks still come first, and M == 0 launches nothing
    with pytest.raises(B.SwigluError) as e:
        B.swiglu_mlp_unfused_static(A_, W1_, W2_, Y_, M=16, N=4860, K=896, stream=0)
    assert e.value.status == B.SWIGLU_ERR_UNSUPPORTED
    B.swiglu_mlp_unfused_static(A_, W1_, W2_, Y_, M=0, N=4864, K=896, stream=0)


@pytest.mark.gpu
def test_static_scratch_entry_point_matches_the_existing_path_on_two_calls_in_a_row():
    import torch
    import oracle
    from paper_2607_02521_b200 import check, inputs

    assert torch.cuda.is_available(), "GPU tests need a B200"
    B.load()

    def dev(bits):
        return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).cuda().view(torch.bfloat16)

    def host(t):
        return t.view(torch.int16).cpu().numpy().view(np.uint16)

    # two calls in a row on the same (shared) scratch: a large-M call through the pair GEMMs with
    # ragged M / N / K, then a SMALLER decode-sized call through the merged Gate|Up kernel, whose
    # scratch region still holds the first call's Gate / Up; then the first shape again
    shapes = [(700, 1160, 328, 901), (16, 4864, 896, 902), (700, 1160, 328, 903)]
    for M, N, K, seed in shapes:
        A, W1, W2 = inputs.make_case(M, N, K, seed=seed, std=0.05)
        dA, dW1, dW2 = dev(A), dev(W1), dev(W2)
        y_new = torch.full((M, N), float("nan"), dtype=torch.bfloat16, device="cuda")
        B.swiglu_mlp_unfused_static(dA, dW1, dW2, y_new)
        torch.cuda.synchronize()
        y_old = torch.full((M, N), float("nan"), dtype=torch.bfloat16, device="cuda")
        B.swiglu_mlp_unfused(dA, dW1, dW2, y_old)
        torch.cuda.synchronize()
        new = inputs.bf16_bits_to_f64(host(y_new))
        old = inputs.bf16_bits_to_f64(host(y_old))
        assert np.all(np.isfinite(new)), (M, N, K)
        assert np.all(np.abs(new - old) <= ATOL + RTOL * np.abs(old)), (M, N, K)
        assert np.array_equal(host(y_new), host(y_old)), (M, N, K)   # same kernels, same order
        y_ref, _ = oracle.swiglu_oracle(A, W1, W2)
        rep = check.compare(host(y_new), y_ref)
        assert rep.mismatches == 0, ((M, N, K), rep)

    # beyond the array: rejected with its own code, nothing launched, Y untouched
    M, N, K = 2048, 4864, 64      # 2 * 2048 * 4864 * 2 = 38 MiB > 32 MiB
    A, W1, W2 = inputs.make_case(M, N, K, seed=904, std=0.05)
    y = torch.full((M, N), float("nan"), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(B.SwigluError) as e:
        B.swiglu_mlp_unfused_static(dev(A), dev(W1), dev(W2), y)
    assert e.value.status == B.SWIGLU_ERR_WORKSPACE
    torch.cuda.synchronize()
    assert bool(torch.isnan(y.float()).all())
