"""Pins of the oracle's weight interleave (oracle.pack_weights; PAPER.md lines 159, 167-169:
Kernel-2 "interleaves W1 and W2", a one-time preprocessing step; R18 for the layout
reading).  Index work, so everything is bit-exact."""
import os

import numpy as np
import pytest

import oracle

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "pack_example.txt")


def tagged(K, N, which):
    """Every element carries its own identity: bits = which*0x8000 + (k*N + n) (< 0x8000)."""
    assert K * N < 0x8000
    return (np.arange(K * N, dtype=np.uint16).reshape(K, N) + np.uint16(which * 0x8000))


@pytest.mark.parametrize("K,N", [(1, 8), (3, 64), (5, 72), (2, 128), (7, 136), (4, 264), (2, 384)])
def test_every_weight_appears_exactly_once_at_the_stated_place(K, N):
    W1, W2 = tagged(K, N, 0), tagged(K, N, 1)
    Wp = oracle.pack_weights(W1, W2)
    T = (N + 127) // 128
    Kp = oracle.pack_rows(K)
    assert Wp.shape == (T, 4, Kp, 64)
    assert Kp - K in (8, 16) and (Kp * 128 // 1024) % 2 == 1 if K % 8 == 0 else Kp > K
    # inverse walk, written from the other side: for each (matrix, k, n) say where it must be
    seen = np.zeros(Wp.shape, dtype=bool)
    for which, W in ((0, W1), (1, W2)):
        for k in range(K):
            for n in range(N):
                t, r = divmod(n, 128)
                half, c = divmod(r, 64)
                s = 2 * half + which                  # gate 0, up 0, gate 1, up 1
                assert Wp[t, s, k, c] == W[k, n]
                assert not seen[t, s, k, c]
                seen[t, s, k, c] = True
    assert seen.sum() == 2 * K * N
    assert np.all(Wp[~seen] == 0)                     # padding columns (n >= N) and rows (k >= K)


def test_gate_and_up_columns_of_one_output_share_a_tile():
    """The property the interleave exists for: output column n's Gate and
    Up weights are neighbours -- same 128-column tile, adjacent slabs, same (k, c)."""
    K, N = 3, 200
    W1, W2 = tagged(K, N, 0), tagged(K, N, 1)
    Wp = oracle.pack_weights(W1, W2)
    for n in range(N):
        t, r = divmod(n, 128)
        half, c = divmod(r, 64)
        assert np.array_equal(Wp[t, 2 * half, :K, c], W1[:, n])
        assert np.array_equal(Wp[t, 2 * half + 1, :K, c], W2[:, n])


@pytest.mark.parametrize("K,Kp", [(8, 24), (16, 24), (896, 904), (1536, 1544), (3584, 3592), (5120, 5128),
                                  (8192, 8200), (72, 88)])
def test_slab_pitch_is_an_odd_number_of_kib(K, Kp):
    """Hand-computed: K/8 even -> +8 rows, K/8 odd -> +16, so Kp * 128 B is an odd multiple of 1 KiB."""
    assert oracle.pack_rows(K) == Kp
    assert (Kp * 128) % 1024 == 0 and ((Kp * 128) // 1024) % 2 == 1


def test_hand_written_example():
    """tests/golden/pack_example.txt: K = 1, N = 136 written out by hand from the definition."""
    rows = [l.split() for l in open(GOLDEN) if l.strip() and not l.startswith("#")]
    K, N = 1, 136
    W1 = (np.arange(N, dtype=np.uint16) + 1000).reshape(K, N)
    W2 = (np.arange(N, dtype=np.uint16) + 2000).reshape(K, N)
    Wp = oracle.pack_weights(W1, W2)
    for t, s, c, value in rows:
        assert int(Wp[int(t), int(s), 0, int(c)]) == int(value), (t, s, c)
