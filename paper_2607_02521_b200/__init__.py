"""B200-native fused gated MLP  Y = SiLU(A.W1) (.) (A.W2)  (arxiv/paper_2607_02521).

The product is the C-ABI library ``libswiglu_b200.so`` (include/swiglu_mlp.h) built from
``csrc/``; ``binding`` is the thin ctypes layer over it with the same names.  Importing the
package does not load the library (``inputs`` and ``check`` are usable on a CPU-only host);
the first call into ``binding`` does, and raises if the library is missing.
"""
__all__ = ["inputs", "check"]
