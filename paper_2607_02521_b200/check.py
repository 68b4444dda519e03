"""Harness-side comparison of a bf16 result with an fp64 reference.

The bound is BASELINE.json north_star's: an output is a MISMATCH when it is non-finite or
|y - y_ref| > 2e-3 + 1.6e-2*|y_ref| (two bf16 ulps relative plus an absolute floor).  This
is comparison bookkeeping only; none of the method's arithmetic is here and the reference
values are passed in by the caller (tests / bench), never computed here.
"""
from __future__ import annotations

from dataclasses import dataclass, asdict

import numpy as np

from .inputs import bf16_bits_to_f64, f32_to_bf16_bits

ATOL = 2e-3
RTOL = 1.6e-2


@dataclass
class Report:
    checked: int          # elements compared
    mismatches: int       # elements outside the bound (or non-finite)
    max_abs_err: float
    max_ratio: float      # max |err| / (ATOL + RTOL*|y_ref|); <= 1 means inside the bound
    not_rne_of_ref: int   # elements != bf16_RNE(y_ref)  (secondary statistic, R9)

    def as_dict(self):
        return asdict(self)


def compare(y_bits: np.ndarray, y_ref: np.ndarray) -> Report:
    """y_bits: bf16 bit patterns (uint16) from the GPU; y_ref: fp64 reference, same shape."""
    y_bits = np.ascontiguousarray(y_bits, dtype=np.uint16)
    y_ref = np.ascontiguousarray(y_ref, dtype=np.float64)
    if y_bits.shape != y_ref.shape:
        raise ValueError(f"shape mismatch {y_bits.shape} vs {y_ref.shape}")
    if y_bits.size == 0:
        return Report(0, 0, 0.0, 0.0, 0)
    y = bf16_bits_to_f64(y_bits)
    err = np.abs(y - y_ref)
    bound = ATOL + RTOL * np.abs(y_ref)
    bad = ~np.isfinite(y) | (err > bound)
    finite_err = np.where(np.isfinite(err), err, np.inf)
    ref_bits = f32_to_bf16_bits(y_ref.astype(np.float32))
    # +0 and -0 are the same value: compare through the decoded numbers
    not_rne = int(np.count_nonzero(bf16_bits_to_f64(ref_bits) != y))
    return Report(
        checked=int(y.size),
        mismatches=int(np.count_nonzero(bad)),
        max_abs_err=float(finite_err.max()),
        max_ratio=float((finite_err / bound).max()),
        not_rne_of_ref=not_rne,
    )
