"""CPU-side checks of the C-ABI boundary (no GPU needed): the library builds for sm_100a, loads, exports every
symbol include/vla_ternary.h declares, and its host-side argument validation answers before any launch."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "vla_ternary.h")


@pytest.fixture(scope="module")
def vla():
    from paper_2606_08094_b200 import binding
    return binding


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b(vla_[a-z0-9_]+)\s*\(", src)
    return sorted(set(names))


def test_header_declares_the_north_star_calls():
    names = _declared_functions()
    for required in ("vla_ternary_pack", "vla_act_quant", "vla_ternary_gemm", "vla_ternary_linear",
                     "vla_ternary_unpack", "vla_ternary_packed_bytes", "vla_ternary_workspace_bytes"):
        assert required in names


def test_library_exports_every_declared_symbol(vla):
    lib = ctypes.CDLL(vla.LIB_PATH)
    for name in _declared_functions():
        assert hasattr(lib, name), name
    assert sorted(vla.EXPORTS) == _declared_functions()


def test_packed_bytes_is_a_quarter_byte_per_weight(vla):
    # "four two-bit codes per byte": no padding at supported shapes
    for K, N in [(256, 256), (2560, 2560), (2560, 640), (2560, 6912), (6912, 2560), (8192, 8192)]:
        assert vla.vla_ternary_packed_bytes(N, K) == N * K // 4
    assert vla.vla_ternary_packed_bytes(100, 256) == 0
    assert vla.vla_ternary_packed_bytes(256, 100) == 0
    assert vla.vla_ternary_packed_bytes(0, 256) == 0


def test_workspace_bytes(vla):
    for M, N, K in [(1, 256, 256), (8, 2560, 2560), (544, 2560, 6912)]:
        ws = vla.vla_ternary_workspace_bytes(M, N, K)
        assert ws % 256 == 0 and ws >= M * K + 4 * M
        hs = vla.vla_ternary_host_workspace_bytes(M, N, K, vla.VLA_F32)
        assert hs >= ws + 2 * M * K + 4 * M * N
    assert vla.vla_ternary_workspace_bytes(0, 256, 256) == 0
    assert vla.vla_ternary_workspace_bytes(8, 100, 256) == 0


def test_status_strings(vla):
    seen = set()
    for s in range(0, 9):
        t = vla.vla_status_string(s)
        assert t and t not in seen
        seen.add(t)
    assert vla.vla_status_string(0) == "VLA_OK"


def test_host_validation_precedes_any_launch(vla):
    """NULL / shape / dtype / alignment errors are reported from the host, GPU or not."""
    L = vla._lib
    fake = 0x1000  # 16-byte aligned non-NULL "pointer"; never dereferenced because validation fails first
    assert L.vla_ternary_pack(None, 256, 256, fake, 16384, None) == vla.VLA_ERR_NULL
    assert L.vla_ternary_pack(fake, 100, 256, fake, 16384, None) == vla.VLA_ERR_SHAPE
    assert L.vla_ternary_pack(fake, 256, 256, fake, 100, None) == vla.VLA_ERR_WORKSPACE      # packed buffer too small
    assert L.vla_ternary_pack(fake + 4, 256, 256, fake, 16384, None) == vla.VLA_ERR_ALIGN
    assert L.vla_act_quant(None, 8, 256, fake, fake, None) == vla.VLA_ERR_NULL
    assert L.vla_act_quant(fake, 0, 256, fake, fake, None) == vla.VLA_ERR_SHAPE
    assert L.vla_act_quant(fake, 8, 200, fake, fake, None) == vla.VLA_ERR_SHAPE
    assert L.vla_act_quant(fake, 8, 256, fake + 1, fake, None) == vla.VLA_ERR_ALIGN
    assert L.vla_ternary_gemm(fake, fake, fake, fake, 8, 256, 256, fake, 7, 0, None, 0, None) == vla.VLA_ERR_DTYPE
    assert L.vla_ternary_gemm(fake, fake, fake, fake, 8, 256, 256, fake, 0, 9, None, 0, None) == vla.VLA_ERR_DTYPE
    assert L.vla_ternary_gemm(None, fake, fake, fake, 8, 256, 256, fake, 0, 0, None, 0, None) == vla.VLA_ERR_NULL
    assert L.vla_ternary_gemm(fake, None, fake, fake, 8, 256, 256, fake, 0, 0, None, 0, None) == vla.VLA_ERR_NULL
    assert L.vla_ternary_gemm(fake, fake, fake, fake, 0, 256, 256, fake, 0, 0, None, 0, None) == vla.VLA_ERR_SHAPE
    assert L.vla_ternary_gemm(fake, fake, fake, fake, 8, 256, 320, fake, 0, 0, None, 0, None) == vla.VLA_ERR_SHAPE
    # M=64 is outside the dp4a path's range
    assert L.vla_ternary_gemm(fake, fake, fake, fake, 64, 256, 256, fake, 0, vla.VLA_PATH_SMALL_ALU,
                              None, 0, None) == vla.VLA_ERR_SHAPE
    assert L.vla_ternary_gemm(fake, fake, fake + 8, fake, 8, 256, 256, fake, 0, 0, None, 0, None) == vla.VLA_ERR_ALIGN
    assert L.vla_ternary_linear(fake, fake, fake, 8, 256, 256, fake, 0, 0, None, None, None, 0,
                                None) == vla.VLA_ERR_WORKSPACE
    assert L.vla_ternary_linear(fake, fake, None, 8, 256, 256, fake, 0, 0, None, None, fake, 1 << 20,
                                None) == vla.VLA_ERR_NULL
    assert L.vla_ternary_linear_host(fake, fake, fake, 8, 256, 256, fake, 0, 0, fake, 16, None) == vla.VLA_ERR_WORKSPACE


def test_no_gpu_means_arch_error_not_a_fallback(vla):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    fake = 0x1000
    assert vla._lib.vla_act_quant(fake, 8, 256, fake, fake, None) == vla.VLA_ERR_ARCH
    assert vla._lib.vla_ternary_gemm(fake, fake, fake, fake, 8, 256, 256, fake, 0, 0, None, 0, None) == vla.VLA_ERR_ARCH


def test_auto_path_table(vla):
    assert vla.vla_ternary_auto_path(1, 2560, 2560) in (vla.VLA_PATH_SMALL_ALU, vla.VLA_PATH_SMALL_TC)
    assert vla.vla_ternary_auto_path(544, 2560, 2560) == vla.VLA_PATH_LARGE
    assert vla.vla_ternary_auto_path(4096, 8192, 8192) == vla.VLA_PATH_LARGE
    # 16 < M <= 32: by (N,K), from the measured per-path cost model (profiles/r01d_path_probe.md)
    for M in (17, 24, 32):
        assert vla.vla_ternary_auto_path(M, 8192, 8192) == vla.VLA_PATH_LARGE
        assert vla.vla_ternary_auto_path(M, 6912, 2560) == vla.VLA_PATH_LARGE
        assert vla.vla_ternary_auto_path(M, 2560, 2560) == vla.VLA_PATH_LARGE
        assert vla.vla_ternary_auto_path(M, 2560, 6912) == vla.VLA_PATH_SMALL_TC
        assert vla.vla_ternary_auto_path(M, 640, 2560) == vla.VLA_PATH_SMALL_TC
    for shape in ((2560, 2560), (640, 2560), (6912, 2560), (2560, 6912), (8192, 8192)):
        assert vla.vla_ternary_auto_path(16, *shape) == vla.VLA_PATH_SMALL_TC
        assert vla.vla_ternary_auto_path(33, *shape) == vla.VLA_PATH_LARGE


def test_product_does_not_import_the_oracle():
    """The product path never routes through oracle/: no file of the package mentions it."""
    pkg = os.path.join(ROOT, "paper_2606_08094_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f), errors="ignore").read()
                assert "import oracle" not in text and "from oracle" not in text and "liboracle" not in text, f


def test_grouped_gemm_validates_on_the_host(vla):
    fake = 0x1000
    arr = vla.make_linears([dict(packed=fake, w_scale=fake, out=fake, N=256, out_dtype=1)])
    L = vla._lib
    assert L.vla_ternary_gemm_grouped(None, 1, fake, fake, 64, 256, 0, None) == vla.VLA_ERR_NULL
    assert L.vla_ternary_gemm_grouped(arr, 0, fake, fake, 64, 256, 0, None) == vla.VLA_ERR_SHAPE
    assert L.vla_ternary_gemm_grouped(arr, 9, fake, fake, 64, 256, 0, None) == vla.VLA_ERR_SHAPE
    assert L.vla_ternary_gemm_grouped(arr, 1, fake, fake, 64, 200, 0, None) == vla.VLA_ERR_SHAPE
    assert L.vla_ternary_gemm_grouped(arr, 1, fake + 4, fake, 64, 256, 0, None) == vla.VLA_ERR_ALIGN
    assert L.vla_ternary_gemm_grouped(arr, 1, fake, None, 64, 256, 0, None) == vla.VLA_ERR_NULL
    bad = vla.make_linears([dict(packed=fake, w_scale=fake, out=fake, N=100, out_dtype=1)])
    assert L.vla_ternary_gemm_grouped(bad, 1, fake, fake, 64, 256, 0, None) == vla.VLA_ERR_SHAPE
