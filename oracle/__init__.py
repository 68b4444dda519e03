"""CPU oracle for Y = SiLU(A.W1) (.) (A.W2)  --  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with, and never
imports, ``paper_2607_02521_b200`` (the CUDA path); the CUDA path never imports it.

The arithmetic lives in ``swiglu_oracle.c`` (plain C, fp64; Eq. 1-3);
this module only compiles that file with gcc and marshals numpy arrays into it.
"""
from .oracle import (  # noqa: F401
    ACTIVATIONS,
    activation,
    build,
    e4m3_to_f64,
    max_threads,
    pack_rows,
    pack_weights,
    silu,
    swiglu_oracle,
    swiglu_oracle_fp8,
    swiglu_oracle_rows,
)
