"""Per-tile timeline of the large-M kernels from a debug build (`-DSWIGLU_TRACE`).

    python -m paper_2607_02521_b200.trace_timeline qwen2.5-1.5b 4096 [--variant 1|5] [--act 0..3] [--chunk 0|1]

Builds a SECOND copy of the library with the `%globaltimer` stamps compiled in (the product
library has none), runs one call of the given (shape, M) after three warm-up calls and prints,
for the leader CTA of the first and of the middle CTA pair, when (microseconds from kernel start)
  * the MMA thread could start a tile, saw its first operands, had issued its last MMA,
  * the epilogue saw the accumulator, and was done with the tile,
  * 256-row kernels: inside chunk `--chunk` of the epilogue -- first barrier, TMEM loads retired,
    second barrier (store issue);
  * super-tile kernel: region 0 / region 1 free, head of row block 0 issued, both accumulator
    commits, both drains.
This is the measurement behind DESIGN.md 5.3b.  Needs a B200; not used by tests or bench.py.
"""
from __future__ import annotations

import argparse
import ctypes
import os
import subprocess
import sys
import tempfile

HERE = os.path.dirname(os.path.abspath(__file__))
STRIDE = 8 + 8 * 32   # kGemmTraceStride in gemm_swiglu_kernel.cuh


def build_trace_library(chunk: int) -> str:
    from . import build as libbuild
    out = os.path.join(tempfile.gettempdir(), f"libswiglu_b200_trace_h{chunk}.so")
    cmd = [libbuild._nvcc(), *libbuild.NVCC_FLAGS, "-DSWIGLU_TRACE", f"-DSWIGLU_TRACE_H={chunk}", "-o", out,
           os.path.join(libbuild.CSRC, "swiglu_api.cu")]
    subprocess.run(cmd, check=True)
    return out


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("shape")
    ap.add_argument("M", type=int)
    ap.add_argument("--variant", type=int, default=-1)
    ap.add_argument("--act", type=int, default=0)
    ap.add_argument("--chunk", type=int, default=0)
    ap.add_argument("--tiles", type=int, default=6)
    args = ap.parse_args()
    import torch
    from . import inputs
    lib = ctypes.CDLL(build_trace_library(args.chunk))
    table = dict(inputs.SHAPES)
    table.update(inputs.PAPER_SHAPES)
    K, N, seed, _ = table[args.shape]
    M = args.M
    g = torch.Generator(device="cuda").manual_seed(seed)
    A = torch.randn((M, K), device="cuda", generator=g).bfloat16()
    W1 = (torch.randn((K, N), device="cuda", generator=g) * 0.02).bfloat16()
    W2 = (torch.randn((K, N), device="cuda", generator=g) * 0.02).bfloat16()
    Y = torch.empty((M, N), dtype=torch.bfloat16, device="cuda")
    p, i64, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int
    lib.swiglu_glu_mlp_ex.argtypes = [p, p, p, p, i64, i64, i64, ci, ci, p]
    lib.swiglu_selected_variant.argtypes = [i64, i64, i64, ci]
    lib.swiglu_variant_name.argtypes, lib.swiglu_variant_name.restype = [ci, ci], ctypes.c_char_p
    lib.swiglu_debug_set_trace.argtypes = [p]
    variant = args.variant if args.variant >= 0 else lib.swiglu_selected_variant(M, N, K, 0)
    name = lib.swiglu_variant_name(0, variant).decode()
    trace = torch.zeros((160, STRIDE), dtype=torch.int64, device="cuda")

    def call():
        rc = lib.swiglu_glu_mlp_ex(A.data_ptr(), W1.data_ptr(), W2.data_ptr(), Y.data_ptr(), M, N, K,
                                   args.act, variant, None)
        if rc:
            sys.exit(f"swiglu_glu_mlp_ex failed with status {rc}")
    for _ in range(3):
        call()
    torch.cuda.synchronize()
    lib.swiglu_debug_set_trace(trace.data_ptr())
    call()
    torch.cuda.synchronize()
    lib.swiglu_debug_set_trace(None)
    t = trace.cpu().numpy()
    t0 = t[:, 0][t[:, 0] > 0].min()
    us = lambda x: f"{(x - t0) / 1e3:8.2f}" if x else "       -"
    print(f"{args.shape} M={M} {name} activation {args.act}: kernel span {(t[:, 2].max() - t0) / 1e3:.2f} us")
    super_tile = "512x128" in name
    for cta in (0, 74):
        r = t[cta]
        print(f"CTA {cta}: entry {us(r[0])}  setup done {us(r[1])}  exit {us(r[2])}")
        for it in range(args.tiles):
            s = r[8 + it * 8: 16 + it * 8]
            if not s.any():
                break
            if super_tile:
                print(f"  tile {it:2d}: region0 free {us(s[0])}  head of block 0 issued {us(s[1])}  region1 free {us(s[2])}"
                      f"  commit0 {us(s[5])}  commit1 {us(s[6])} | drain0 from {us(s[3])}  drain1 from {us(s[7])}  done {us(s[4])}")
            else:
                print(f"  tile {it:2d}: mma start {us(s[0])}  first operands {us(s[1])}  last mma issued {us(s[2])}"
                      f" | epilogue {us(s[3])} ..{us(s[4])} | chunk {args.chunk}: barrier {us(s[5])}  tmem loaded {us(s[6])}"
                      f"  staged {us(s[7])}")


if __name__ == "__main__":
    main()
