"""Pins for the CPU oracle (oracle/swiglu_oracle.c) -- checked against things OTHER than
itself: exact rational brute force, hand-worked examples, SiLU closed forms from 50-digit
decimal arithmetic, an identity that reduces Y to two library matmuls, and invariants.

Each pin names the mistake it is there to catch.  PAPER.md lines 86-94 (Eq. 1-3) define the
computation; PAPER.md prints no numeric example, so no pin comes from a printed value.
"""
import itertools
import os
from decimal import Decimal, getcontext
from fractions import Fraction

import numpy as np
import pytest

import oracle
from paper_2607_02521_b200 import inputs

getcontext().prec = 60
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "worked_examples.txt")


def dec_silu(x: Decimal) -> Decimal:
    """SiLU(x) = x * sigma(x) in 60-digit decimal arithmetic."""
    return x / (1 + (-x).exp())


def bits(x):
    return inputs.f64_to_bf16_bits_exact(np.asarray(x, dtype=np.float64))


# ---------------------------------------------------------------- P2: hand-worked examples
def _parse_golden():
    cases, cur, key = [], None, None
    for line in open(GOLDEN):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        if line.startswith("case"):
            cur, key = {"name": line.split()[1]}, None
        elif line == "end":
            cases.append({k: (np.array(v, dtype=object) if k != "name" else v)
                          for k, v in cur.items()})
            cur = None
        elif line in ("A", "W1", "W2", "G", "U", "Y"):
            key = line
            cur[key] = []
        else:
            cur[key].append(line.split())
    return cases


@pytest.mark.parametrize("case", _parse_golden(), ids=lambda c: c["name"])
def test_hand_worked_examples(case):
    """Catches: transposed operands, W read as [N,K], Gate/Up swapped (SiLU(U)*G), sign."""
    f = lambda m: np.array([[float(x) for x in row] for row in m], dtype=np.float64)
    A, W1, W2 = f(case["A"]), f(case["W1"]), f(case["W2"])
    # the fixture's G and U are hand-derived rationals: check them with exact Fractions
    FA = [[Fraction(x) for x in row] for row in case["A"]]
    for name, W in (("G", case["W1"]), ("U", case["W2"])):
        FW = [[Fraction(x) for x in row] for row in W]
        got = [[sum(FA[m][k] * FW[k][n] for k in range(len(FW))) for n in range(len(FW[0]))]
               for m in range(len(FA))]
        want = [[Fraction(x) for x in row] for row in case[name]]
        assert got == want, name
    # the fixture's Y digits re-derived with decimals from its own G and U
    for m, row in enumerate(case["Y"]):
        for n, ytxt in enumerate(row):
            y50 = dec_silu(Decimal(case["G"][m][n])) * Decimal(case["U"][m][n])
            assert abs(Decimal(ytxt) - y50) <= abs(y50) * Decimal("1e-15") + Decimal("1e-300")
    y, _ = oracle.swiglu_oracle(bits(A), bits(W1), bits(W2))
    want = f(case["Y"])
    np.testing.assert_allclose(y, want, rtol=1e-14, atol=1e-300)


# ---------------------------------------------------------------- P1: exact brute force
@pytest.mark.parametrize("M,N,K", [s for s in itertools.product((1, 2, 3, 5), (1, 3, 8, 17),
                                                                   (1, 2, 5, 17))])
def test_brute_force_rational(M, N, K):
    """Catches: wrong index/stride, a dropped or doubled k term, tails, thread partitioning.
    Dot products in exact rational arithmetic (every bf16 is a dyadic rational), SiLU in
    60-digit decimals."""
    A, W1, W2 = inputs.make_case(M, N, K, seed=1000 + 37 * M + 5 * N + K, std=0.5)
    y, _ = oracle.swiglu_oracle(A, W1, W2, nthreads=3)
    fa = [[Fraction(float(v)) for v in row] for row in inputs.bf16_bits_to_f64(A)]
    f1 = [[Fraction(float(v)) for v in row] for row in inputs.bf16_bits_to_f64(W1)]
    f2 = [[Fraction(float(v)) for v in row] for row in inputs.bf16_bits_to_f64(W2)]
    for m in range(M):
        for n in range(N):
            g = sum(fa[m][k] * f1[k][n] for k in range(K))
            u = sum(fa[m][k] * f2[k][n] for k in range(K))
            gd = Decimal(g.numerator) / Decimal(g.denominator)
            ud = Decimal(u.numerator) / Decimal(u.denominator)
            want = float(dec_silu(gd) * ud)
            assert y[m, n] == pytest.approx(want, rel=1e-13, abs=1e-15), (m, n)


def test_panel_and_thread_tails():
    """N straddling the 256-column panel, more threads than units, one thread."""
    A, W1, W2 = inputs.make_case(3, 600, 40, seed=77, std=0.3)
    y1, t1 = oracle.swiglu_oracle(A, W1, W2, nthreads=1)
    y8, t8 = oracle.swiglu_oracle(A, W1, W2, nthreads=64)
    assert t1 == 1 and 1 <= t8 <= 9
    assert np.array_equal(y1, y8)  # outputs are independent: threading cannot change a bit
    a, w1, w2 = map(inputs.bf16_bits_to_f64, (A, W1, W2))
    g, u = a @ w1, a @ w2
    np.testing.assert_allclose(y1, g / (1 + np.exp(-g)) * u, rtol=1e-12, atol=1e-14)


# ---------------------------------------------------------------- P3: SiLU closed forms
@pytest.mark.parametrize("x", [0.0, 1.0, -1.0, 2.0, -2.0, 0.5, -0.375, 3.0, 10.0, -10.0,
                               40.0, -40.0, 88.0, -88.0, 700.0, -700.0])
def test_silu_closed_forms(x):
    """Catches: sigma(-x) instead of sigma(x), a missing factor x, exp overflow."""
    want = dec_silu(Decimal(x))
    got = oracle.silu(x)
    assert np.isfinite(got)
    assert abs(Decimal(got) - want) <= abs(want) * Decimal("4e-16") + Decimal("1e-320")


def test_silu_limits_named_by_north_star():
    """SiLU(0)=0; SiLU(x)->x for large x; SiLU(x)->0 for very negative x (BASELINE.json)."""
    assert oracle.silu(0.0) == 0.0
    assert oracle.silu(40.0) == 40.0          # 40*(1 - e^-40) rounds to 40 in fp64
    assert oracle.silu(1e4) == 1e4            # no overflow of exp(-x)
    assert oracle.silu(-800.0) == 0.0 and not np.isnan(oracle.silu(-800.0))
    assert -2e-16 < oracle.silu(-40.0) < -1.6e-16
    # global minimum of SiLU: value -0.27846454276107379 at x = -1.2784645427610738
    xs = np.linspace(-3, 0, 30001)
    vals = np.array([oracle.silu(float(v)) for v in xs])
    assert abs(xs[vals.argmin()] - (-1.2784645427610738)) < 2e-4
    assert abs(vals.min() - (-0.27846454276107379)) < 1e-9


def test_silu_through_the_whole_oracle():
    """K=1, A=[[x]], W1=[[1]], W2=[[1]]  =>  Y = SiLU(x)*x, x bf16-exact."""
    for x in (0.0, 1.0, -1.0, 2.0, -2.0, 10.0, -10.0, 40.0, -40.0):
        y, _ = oracle.swiglu_oracle(bits([[x]]), bits([[1.0]]), bits([[1.0]]))
        want = dec_silu(Decimal(x)) * Decimal(x)
        assert abs(Decimal(float(y[0, 0])) - want) <= abs(want) * Decimal("4e-16")


# ------------------------------------------- P4: identity reducing Y to two plain matmuls
def test_identity_reduces_to_library_matmuls():
    """sigma(x)+sigma(-x)=1  =>  SiLU(g)-SiLU(-g)=g, so
    oracle(A,W1,W2) - oracle(A,-W1,W2) = (A.W1) (.) (A.W2): two fp64 library matmuls.
    Catches any error in the two contractions, their pairing and the row/column layout,
    independently of how SiLU is evaluated."""
    A, W1, W2 = inputs.make_case(37, 531, 193, seed=5)
    W1neg = W1 ^ np.uint16(0x8000)  # flip the bf16 sign bit: exact negation
    yp, _ = oracle.swiglu_oracle(A, W1, W2)
    yn, _ = oracle.swiglu_oracle(A, W1neg, W2)
    a, w1, w2 = map(inputs.bf16_bits_to_f64, (A, W1, W2))
    want = (a @ w1) * (a @ w2)
    np.testing.assert_allclose(yp - yn, want, rtol=1e-11, atol=1e-13)


def test_library_cross_check_mid_size():
    """P7: Qwen-2.5-1.5B weights (K=1536, N=8960), 24 rows, against numpy fp64 matmul with a
    different summation order."""
    K, N, seed, _ = inputs.SHAPES["qwen2.5-1.5b"]
    W1, W2 = inputs.make_weights(K, N, seed)
    A = inputs.make_activations(24, K, seed)
    y, _ = oracle.swiglu_oracle(A, W1, W2)
    a, w1, w2 = map(inputs.bf16_bits_to_f64, (A, W1, W2))
    g, u = a @ w1, a @ w2
    want = np.where(g >= 0, g / (1 + np.exp(-np.abs(g))), g * np.exp(-np.abs(g)) / (1 + np.exp(-np.abs(g)))) * u
    np.testing.assert_allclose(y, want, rtol=1e-11, atol=1e-13)
    # sampled-rows entry point returns exactly those rows
    rows = np.array([0, 5, 23, 7])
    ysub, _ = oracle.swiglu_oracle_rows(A, W1, W2, rows)
    assert np.array_equal(ysub, y[rows])


# ---------------------------------------------------------------- P5: invariants
def test_zero_activations_give_zero():
    """A = 0 => Y = 0 exactly (BASELINE.json north_star)."""
    _, W1, W2 = inputs.make_case(4, 300, 64, seed=9)
    y, _ = oracle.swiglu_oracle(np.zeros((4, 64), np.uint16), W1, W2)
    assert np.all(y == 0.0)


def test_equal_weights_give_g_times_silu_g():
    """W2 = W1 => Y = SiLU(G)*G = G^2*sigma(G) >= 0 (BASELINE.json north_star); G from a
    library matmul.  Catches Gate/Up cross-wiring and a sign error in sigma."""
    A, W1, _ = inputs.make_case(9, 257, 96, seed=11, std=0.2)
    y, _ = oracle.swiglu_oracle(A, W1, W1)
    assert np.all(y >= 0.0)
    g = inputs.bf16_bits_to_f64(A) @ inputs.bf16_bits_to_f64(W1)
    np.testing.assert_allclose(y, g * g / (1 + np.exp(-g)), rtol=1e-11, atol=1e-14)


def test_gate_and_up_are_not_interchangeable():
    """SiLU acts on A.W1, not on A.W2: swapping W1 and W2 must change Y."""
    A, W1, W2 = inputs.make_case(5, 64, 32, seed=13, std=0.5)
    y12, _ = oracle.swiglu_oracle(A, W1, W2)
    y21, _ = oracle.swiglu_oracle(A, W2, W1)
    assert np.abs(y12 - y21).max() > 1e-3
    # and the difference is what SiLU(g)u - SiLU(u)g predicts: g*u*(sigma(g)-sigma(u))
    a, w1, w2 = map(inputs.bf16_bits_to_f64, (A, W1, W2))
    g, u = a @ w1, a @ w2
    sig = lambda t: 1 / (1 + np.exp(-t))
    np.testing.assert_allclose(y12 - y21, g * u * (sig(g) - sig(u)), rtol=1e-9, atol=1e-13)


# ---------------------------------------------------------------- P6: exact structure
def test_linearity_in_up_permutations_and_prefix():
    A, W1, W2 = inputs.make_case(6, 70, 48, seed=17, std=0.25)
    y, _ = oracle.swiglu_oracle(A, W1, W2)
    # doubling W2 is exact in bf16 (exponent + 1) and doubles Y exactly
    W2x2 = (W2 + np.uint16(0x0080)).astype(np.uint16)
    assert np.array_equal(inputs.bf16_bits_to_f64(W2x2), 2 * inputs.bf16_bits_to_f64(W2))
    y2, _ = oracle.swiglu_oracle(A, W1, W2x2)
    assert np.array_equal(y2, 2 * y)
    # row permutation of A permutes rows of Y; joint column permutation permutes columns
    rp = np.random.default_rng(0).permutation(6)
    cp = np.random.default_rng(1).permutation(70)
    yr, _ = oracle.swiglu_oracle(A[rp], W1, W2)
    assert np.array_equal(yr, y[rp])
    yc, _ = oracle.swiglu_oracle(A, W1[:, cp], W2[:, cp])
    assert np.array_equal(yc, y[:, cp])
    # prefix property in M (what lets the bench slice A = A_max[:M])
    yp, _ = oracle.swiglu_oracle(A[:2], W1, W2)
    assert np.array_equal(yp, y[:2])


def test_empty_and_degenerate_shapes():
    y, _ = oracle.swiglu_oracle(np.zeros((0, 8), np.uint16), np.zeros((8, 16), np.uint16),
                                np.zeros((8, 16), np.uint16))
    assert y.shape == (0, 16)
    # K = 0: empty sums, G = U = 0, Y = SiLU(0)*0 = 0
    y, _ = oracle.swiglu_oracle(np.zeros((2, 0), np.uint16), np.zeros((0, 3), np.uint16),
                                np.zeros((0, 3), np.uint16))
    assert y.shape == (2, 3) and np.all(y == 0.0)
