"""Pins for the oracle's other gated activations (GeGLU, ReGLU; PAPER.md line 56 and line 392
item 4) -- again against things other than the oracle: 60-digit decimal evaluation of the
textbook definitions (erf from its Maclaurin series, tanh from exp), the printed value of the
standard normal CDF at 1, the odd-part identity act(x) - act(-x) = x that reduces Y to two
library matmuls, and limits.  SiLU (act 0) is pinned in test_oracle_pins.py.
"""
from decimal import Decimal, getcontext

import numpy as np
import pytest

import oracle
from paper_2607_02521_b200 import inputs

getcontext().prec = 60
PI = Decimal("3.14159265358979323846264338327950288419716939937510582097494")


def dec_erf(x: Decimal) -> Decimal:
    """erf(x) = 2/sqrt(pi) * sum_n (-1)^n x^(2n+1) / (n! (2n+1)), summed until it stops moving
    (fine for |x| <= 6 at 60 digits plus guard digits)."""
    getcontext().prec = 120
    term, total, n = x, x, 0
    while abs(term) > Decimal(10) ** -100:
        n += 1
        term = -term * x * x / n
        total += term / (2 * n + 1)
    out = 2 * total / PI.sqrt()
    getcontext().prec = 60
    return +out


def dec_tanh(x: Decimal) -> Decimal:
    e = (2 * x).exp()
    return (e - 1) / (e + 1)


def dec_act(act: str, x: Decimal) -> Decimal:
    if act == "gelu":        # x * Phi(x), Phi(x) = (1 + erf(x / sqrt 2)) / 2
        return x * (1 + dec_erf(x / Decimal(2).sqrt())) / 2
    if act == "gelu_tanh":   # 0.5 x (1 + tanh(sqrt(2/pi) (x + 0.044715 x^3)))
        u = (2 / PI).sqrt() * (x + Decimal("0.044715") * x ** 3)
        return x * (1 + dec_tanh(u)) / 2
    if act == "relu":
        return max(x, Decimal(0))
    raise ValueError(act)


XS = [0.0, 1.0, -1.0, 0.5, -0.375, 2.0, -2.0, 3.0, -3.0, 5.0, -5.0]


@pytest.mark.parametrize("act", ["gelu", "gelu_tanh", "relu"])
@pytest.mark.parametrize("x", XS)
def test_activation_closed_forms(act, x):
    """Catches: Phi(-x) for Phi(x), a missing factor 1/2 or x, the cubic coefficient, erf's
    argument not divided by sqrt 2, cancellation in the negative tail."""
    want = dec_act(act, Decimal(x))
    got = oracle.activation(act, x)
    # a few fp64 roundings (erfc / tanh, the products; 0.044715 held as a double)
    tol = Decimal("1e-14")   # glibc erfc is good to ~10 ulp in the tail
    assert abs(Decimal(got) - want) <= abs(want) * tol + Decimal("1e-300"), (act, x, got, want)


def test_printed_values_and_limits():
    # standard normal CDF at 1 (any table): Phi(1) = 0.8413447460685429...
    assert abs(oracle.activation("gelu", 1.0) - 0.8413447460685429) < 1e-15
    assert abs(oracle.activation("gelu", -1.0) - (-0.15865525393145707)) < 1e-15
    for act in ("gelu", "gelu_tanh", "relu"):
        assert oracle.activation(act, 0.0) == 0.0
        assert oracle.activation(act, 40.0) == 40.0           # act(x) -> x
        assert abs(oracle.activation(act, -40.0)) < 1e-300    # act(x) -> 0 (0- allowed)
        assert not np.isnan(oracle.activation(act, -1e4))
    # GELU's negative tail keeps its relative accuracy: x*Phi(x) at -8 is -4.98e-15
    want = float(dec_act("gelu", Decimal(-8)))
    assert -4.98e-15 < want < -4.97e-15
    assert abs(oracle.activation("gelu", -8.0) / want - 1) < 1e-13
    # ReLU is exact
    assert oracle.activation("relu", -3.5) == 0.0 and oracle.activation("relu", 3.5) == 3.5
    # the two GELU forms differ (by < 5e-4) -- they are not the same function
    d = abs(oracle.activation("gelu", 2.0) - oracle.activation("gelu_tanh", 2.0))
    assert 1e-5 < d < 5e-4


@pytest.mark.parametrize("act", ["gelu", "gelu_tanh", "relu"])
def test_odd_part_identity_reduces_to_library_matmuls(act):
    """Phi(x)+Phi(-x)=1, tanh odd, relu(x)-relu(-x)=x  =>  act(g)-act(-g)=g for all three, so
    oracle(A,W1,W2) - oracle(A,-W1,W2) = (A.W1)(.)(A.W2): two library fp64 matmuls.  Catches a
    wrong operand, pairing or layout on the activation-dispatch path."""
    A, W1, W2 = inputs.make_case(19, 300, 129, seed=6, std=0.2)
    W1neg = W1 ^ np.uint16(0x8000)
    yp, _ = oracle.swiglu_oracle(A, W1, W2, act=act)
    yn, _ = oracle.swiglu_oracle(A, W1neg, W2, act=act)
    a, w1, w2 = map(inputs.bf16_bits_to_f64, (A, W1, W2))
    np.testing.assert_allclose(yp - yn, (a @ w1) * (a @ w2), rtol=1e-11, atol=1e-13)


@pytest.mark.parametrize("act", ["gelu", "gelu_tanh", "relu"])
def test_whole_oracle_against_decimal_and_rows_form(act):
    """Y = act(G) * U element by element from library-matmul G, U and the decimal activation;
    the sampled-rows entry point returns exactly those rows; act 0 is still the default."""
    A, W1, W2 = inputs.make_case(5, 40, 24, seed=9, std=0.3)
    y, _ = oracle.swiglu_oracle(A, W1, W2, act=act)
    a, w1, w2 = map(inputs.bf16_bits_to_f64, (A, W1, W2))
    g, u = a @ w1, a @ w2
    for m in range(5):
        for n in range(0, 40, 7):
            want = float(dec_act(act, Decimal(float(g[m, n]))) * Decimal(float(u[m, n])))
            assert y[m, n] == pytest.approx(want, rel=1e-12, abs=1e-15)
    rows = np.array([4, 0, 2])
    ysub, _ = oracle.swiglu_oracle_rows(A, W1, W2, rows, act=act)
    assert np.array_equal(ysub, y[rows])
    y0, _ = oracle.swiglu_oracle(A, W1, W2)
    ysilu, _ = oracle.swiglu_oracle(A, W1, W2, act="silu")
    assert np.array_equal(y0, ysilu) and not np.array_equal(y0, y)


def test_relu_gives_exact_zeros_where_gate_is_negative():
    A, W1, W2 = inputs.make_case(8, 64, 32, seed=11, std=0.3)
    y, _ = oracle.swiglu_oracle(A, W1, W2, act="relu")
    a, w1 = inputs.bf16_bits_to_f64(A), inputs.bf16_bits_to_f64(W1)
    neg = (a @ w1) < -1e-9
    assert neg.any() and np.all(y[neg] == 0.0)
