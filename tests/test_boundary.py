"""Host logic of the C-ABI boundary, no GPU needed: the library loads, exports every symbol
include/swiglu_mlp.h declares, and rejects bad arguments before any CUDA call."""
import os
import re

import pytest

from paper_2607_02521_b200 import binding as B
from paper_2607_02521_b200 import build as libbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    libbuild.build()
    return B.load()


def test_every_declared_symbol_is_exported(lib):
    header = open(os.path.join(ROOT, "include", "swiglu_mlp.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(swiglu_[a-z0-9_]+)\s*\(", header))
    assert declared == set(B.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_version_status_strings_and_variant_table(lib):
    assert "sm_100a" in B.swiglu_version()
    assert B.status_string(0) == "SWIGLU_OK" and B.status_string(5) == "SWIGLU_ERR_ALIASING"
    nf, nu = B.swiglu_num_variants(False), B.swiglu_num_variants(True)
    assert nf >= 3 and nu >= 1
    names = [B.swiglu_variant_name(v) for v in range(nf)]
    assert len(set(names)) == nf and all(names)
    assert B.swiglu_variant_name(nf) is None and B.swiglu_variant_name(-1) is None
    # dispatch is a host-side table: decode sizes go to the swap-AB kernel, large M does not
    small = B.swiglu_variant_name(B.swiglu_selected_variant(16, 4864, 896))
    large = B.swiglu_variant_name(B.swiglu_selected_variant(4096, 8960, 1536))
    assert "smallm" in small and "smallm" not in large
    assert B.swiglu_launches_per_call(16, 4864, 896) == 1
    assert B.swiglu_launches_per_call(16, 4864, 896, unfused=True) == 2     # merged Gate|Up GEMM
    assert B.swiglu_launches_per_call(4096, 8960, 1536, unfused=True) == 3  # two GEMMs + elementwise
    assert "smallm" in B.swiglu_variant_name(B.swiglu_selected_variant(16, 4864, 896, unfused=True),
                                             unfused=True)
    assert B.swiglu_launches_per_call(0, 4864, 896) == 0


def test_large_m_dispatch_table(lib):
    """Host-only table (no CUDA call): the 512-row super tile for M > 512 with K >= 768 where its
    wave efficiency is within 3 points of the 256-row pair kernel's, the pair kernel otherwise
    (profiles/r02b_variant_sweep_super_tile.md); same rule for the unfused GEMM."""
    name = lambda M, N, K, unfused=False: B.swiglu_variant_name(
        B.swiglu_selected_variant(M, N, K, unfused=unfused), unfused=unfused)
    for K, N in ((3584, 18944), (5120, 27648), (8192, 29568), (5120, 13824)):
        for M in (1024, 2048, 4096, 8192):
            assert "512x128" in name(M, N, K), (M, N, K)
            assert "512x256" in name(M, N, K, unfused=True), (M, N, K)
        for M in (129, 256, 512, 768):
            assert name(M, N, K) == "fused_2cta_256x128", (M, N, K)
        for M in (300, 384, 600, 640):     # three / five 128-row tiles: no padded half tile row
            assert name(M, N, K) == "fused_1cta_128x128", (M, N, K)
    for K, N in ((896, 4864), (1536, 8960)):            # short K too, from M = 1024 up
        for M in (1024, 4096, 8192):
            assert "512x128" in name(M, N, K), (M, N, K)
        for M in (256, 512, 768):
            assert name(M, N, K) == "fused_2cta_256x128", (M, N, K)
    assert name(4096, 4864, 512) == "fused_2cta_256x128"   # fewer than 12 k-blocks per tile
    # no workspace for the super tile (its last wave is cut into row-block / quarter units, not in K)
    assert B.swiglu_workspace_bytes(8192, 29568, 8192, unfused=False) == 0
    assert B.swiglu_workspace_bytes(512, 29568, 8192, unfused=False) > 0     # pair kernel, K-split tail


def test_activation_table(lib):
    assert [B.swiglu_activation_name(i) for i in range(5)] == ["silu", "gelu", "gelu_tanh", "relu", None]
    assert B.ACTIVATIONS == {"silu": 0, "gelu": 1, "gelu_tanh": 2, "relu": 3}
    # validation precedes any CUDA call for the activation entry points too
    rc = lib.swiglu_glu_mlp(0x10000000, 0x20000000, 0x30000000, 0x40000000, 4, 12, 8, 0, None)
    assert rc == B.SWIGLU_ERR_UNSUPPORTED            # N % 8 != 0
    rc = lib.swiglu_glu_mlp(0x10000000, 0x20000000, 0x30000000, 0x40000000, 4, 16, 8, 7, None)
    assert rc == B.SWIGLU_ERR_UNSUPPORTED            # unknown activation
    assert lib.swiglu_act_mul(0x10, 0x20, 0x30, 16, 5, None) == B.SWIGLU_ERR_UNSUPPORTED


def test_env_overrides_are_read_once_and_on_reload(lib, monkeypatch):
    """The hot path does no getenv: an override set after the first call is invisible until
    swiglu_reload_env()."""
    auto = B.swiglu_selected_variant(4096, 8960, 1536)
    monkeypatch.setenv("SWIGLU_VARIANT", "0")
    assert B.swiglu_selected_variant(4096, 8960, 1536) == auto      # not re-read
    B.swiglu_reload_env()
    assert B.swiglu_selected_variant(4096, 8960, 1536) == 0
    monkeypatch.delenv("SWIGLU_VARIANT")
    B.swiglu_reload_env()
    assert B.swiglu_selected_variant(4096, 8960, 1536) == auto


def test_tensor_map_cache_stats_are_callable_without_a_device(lib):
    hits, misses, slots = B.swiglu_tensor_map_cache_stats()
    assert slots >= 64 and hits >= 0 and misses >= 0


def test_workspace_query(lib):
    assert B.swiglu_workspace_bytes(128, 8960, 1536, unfused=False) == 0
    need = B.swiglu_workspace_bytes(128, 8960, 1536, unfused=True)
    assert need >= 2 * 128 * 8960 * 2 and need % 256 == 0
    assert B.swiglu_workspace_bytes(-1, 8, 8, unfused=True) == 0


A, W1, W2, Y = 0x10000000, 0x20000000, 0x30000000, 0x40000000  # fake, aligned, disjoint


@pytest.mark.parametrize("args,code", [
    ((A, W1, W2, Y, 16, 4864, 896), B.SWIGLU_OK),
    ((None, None, None, None, 0, 4864, 896), B.SWIGLU_OK),               # M == 0: nothing to do
    ((None, W1, W2, Y, 16, 4864, 896), B.SWIGLU_ERR_NULL_POINTER),
    ((A, W1, W2, None, 16, 4864, 896), B.SWIGLU_ERR_NULL_POINTER),
    ((A, W1, W2, Y, -1, 4864, 896), B.SWIGLU_ERR_BAD_SHAPE),
    ((A, W1, W2, Y, 16, 0, 896), B.SWIGLU_ERR_BAD_SHAPE),
    ((A, W1, W2, Y, 16, 4864, 0), B.SWIGLU_ERR_BAD_SHAPE),
    ((A, W1, W2, Y, 2**40, 2**30, 2**30), B.SWIGLU_ERR_BAD_SHAPE),       # byte count overflow
    ((A, W1, W2, Y, 16, 4860, 896), B.SWIGLU_ERR_UNSUPPORTED),           # N % 8
    ((A, W1, W2, Y, 16, 4864, 900), B.SWIGLU_ERR_UNSUPPORTED),           # K % 8
    ((A + 2, W1, W2, Y, 16, 4864, 896), B.SWIGLU_ERR_MISALIGNED),
    ((A, W1, W2, Y + 8, 16, 4864, 896), B.SWIGLU_ERR_MISALIGNED),
    ((A, W1, W2, A, 16, 4864, 896), B.SWIGLU_ERR_ALIASING),              # Y == A
    ((A, W1, W2, W2 + 4864 * 2 * 10, 16, 4864, 896), B.SWIGLU_ERR_ALIASING),  # Y inside W2
    ((A, W1, W2, A - 16 * 4864 * 2 + 16, 16, 4864, 896), B.SWIGLU_ERR_ALIASING),  # Y tail hits A
])
def test_validation_codes(lib, args, code):
    assert B.swiglu_validate(*args) == code
    if code != B.SWIGLU_OK:
        assert B.last_error()


def test_compute_entry_points_validate_before_touching_cuda(lib):
    """Bad arguments come back with their own code even on a host without a GPU."""
    for fn in (B.swiglu_mlp, B.swiglu_mlp_unfused):
        with pytest.raises(B.SwigluError) as e:
            fn(A, W1, W2, Y, M=16, N=4860, K=896, stream=0)
        assert e.value.status == B.SWIGLU_ERR_UNSUPPORTED
        fn(A, W1, W2, Y, M=0, N=4864, K=896, stream=0)  # M == 0: OK, launches nothing
    with pytest.raises(B.SwigluError) as e:
        B.swiglu_mlp_ex(A, W1, W2, Y, M=16, N=4864, K=896, variant=99, stream=0)
    assert e.value.status == B.SWIGLU_ERR_UNSUPPORTED
    with pytest.raises(B.SwigluError) as e:
        B.swiglu_mlp_unfused_ex(A, W1, W2, Y, M=16, N=4864, K=896, workspace=None,
                                workspace_bytes=0, stream=0)
    assert e.value.status == B.SWIGLU_ERR_WORKSPACE


def test_no_cpu_fallback_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(B.SwigluError) as e:
        B.swiglu_mlp(A, W1, W2, Y, M=16, N=4864, K=896, stream=0)
    assert e.value.status in (B.SWIGLU_ERR_CUDA, B.SWIGLU_ERR_ARCH)


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_02521_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.replace("the oracle", "").replace("oracle's", "") \
                    or f in ("inputs.py", "check.py"), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2607_02521_b200" not in text
            assert "from paper_2607_02521_b200" not in text


def test_header_is_plain_c_and_the_library_links_from_c(tmp_path):
    """include/swiglu_mlp.h compiles as C11 (no C++ or torch types) and a C program linked
    against the shared library can call the host-only entry points."""
    import subprocess
    src = tmp_path / "abi.c"
    src.write_text(r"""
#include <stdio.h>
#include "swiglu_mlp.h"
int main(void) {
  printf("%s\n", swiglu_version());
  printf("%d %d\n", swiglu_num_variants(0), swiglu_num_variants(1));
  printf("%s\n", swiglu_variant_name(0, swiglu_selected_variant(16, 4864, 896, 0)));
  printf("%d\n", swiglu_validate((void*)16, (void*)32, (void*)48, (void*)64, 4, 12, 8));
  printf("%d\n", swiglu_mlp(0, 0, 0, 0, 0, 16, 8, 0));          /* M == 0: OK, no launch */
  printf("%s\n", swiglu_activation_name(SWIGLU_ACT_GELU_TANH));
  printf("%zu\n", swiglu_workspace_bytes(128, 8960, 1536, 1, -1));
  return 0;
}
""")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    pkg = os.path.join(root, "paper_2607_02521_b200")
    exe = tmp_path / "abi"
    subprocess.run(["gcc", "-std=c11", "-Wall", "-Wextra", "-Werror", "-pedantic",
                    "-I", os.path.join(root, "include"), str(src), "-o", str(exe),
                    "-L", pkg, "-l:libswiglu_b200.so", f"-Wl,-rpath,{pkg}"], check=True)
    out = subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split("\n")
    assert "sm_100a" in out[0]
    assert out[1].split() == [str(B.swiglu_num_variants(False)), str(B.swiglu_num_variants(True))]
    assert "smallm" in out[2]
    assert int(out[3]) == B.SWIGLU_ERR_UNSUPPORTED and int(out[4]) == B.SWIGLU_OK
    assert out[5] == "gelu_tanh" and int(out[6]) >= 2 * 128 * 8960 * 2
