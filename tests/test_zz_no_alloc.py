"""vla_ternary_linear_static (include/vla_ternary.h, csrc/no_alloc.cu): the entry point that allocates nothing -- its
scratch (quantised activations + scales) is a fixed device array inside the library.  The GPU test checks its output
against the existing path (vla_ternary_linear with a caller workspace) bit for bit -- the bar of test_gpu_parity.py for
these outputs -- on two calls in a row that share the array, for the small-M (IMMA) and the large-M (tcgen05) kernels.
Collected last on purpose (the run is `pytest -x`); passes alone in a fresh process and after the others.
"""
import numpy as np
import pytest
import torch

from paper_2606_08094_b200 import synth


@pytest.fixture(scope="module")
def vla():
    from paper_2606_08094_b200 import binding
    return binding


FAKE = 0x10000   # aligned non-NULL "pointer"; never dereferenced: the size check comes before any CUDA call


def test_static_limit_is_enforced_on_the_host(vla):
    L = vla._lib
    over_mk = vla.VLA_STATIC_MAX_MK // 8192 + 1                      # M * 8192 just above the limit
    assert L.vla_ternary_linear_static(FAKE, FAKE, FAKE, over_mk, 256, 8192, FAKE, 0, 0, None) == vla.VLA_ERR_WORKSPACE
    assert L.vla_ternary_linear_static(FAKE, FAKE, FAKE, vla.VLA_STATIC_MAX_M + 1, 256, 128, FAKE, 0, 0, None) == vla.VLA_ERR_WORKSPACE
    assert L.vla_ternary_linear_static(None, FAKE, FAKE, 8, 256, 256, FAKE, 0, 0, None) == vla.VLA_ERR_NULL
    assert L.vla_ternary_linear_static(FAKE, FAKE, FAKE, 0, 256, 256, FAKE, 0, 0, None) == vla.VLA_ERR_SHAPE
    assert "workspace" in vla.vla_status_string(vla.VLA_ERR_WORKSPACE).lower()


def _dev_bf16(bits_u16):
    return torch.from_numpy(np.ascontiguousarray(bits_u16).view(np.int16)).cuda().view(torch.bfloat16)


_TDT = {0: torch.float32, 1: torch.bfloat16, 2: torch.int32}


def _raw(t):
    return t.contiguous().view(torch.uint8).cpu().numpy()


@pytest.mark.gpu
@pytest.mark.parametrize("M,K,N,dtype", [(8, 2560, 640, 1), (16, 6912, 256, 0), (544, 2560, 640, 0), (200, 640, 384, 2)])
def test_static_entry_point_matches_the_workspace_path_twice(vla, M, K, N, dtype):
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    w = synth.ternary_weights(N, K, 0.35, 9700 + M)
    packed = vla.pack_weights(torch.from_numpy(w).cuda())
    beta = torch.tensor([synth.weight_scale(9701 + M)], dtype=torch.float32, device="cuda")
    nb = vla.vla_ternary_workspace_bytes(M, N, K)
    ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
    for call in range(2):                                            # the second call finds the first one's scratch
        x = _dev_bf16(synth.activations(M, K, 9710 + 7 * call + M, outlier_frac=0.01))
        ref = torch.full((M, N), -7, dtype=_TDT[dtype], device="cuda")
        got = torch.full((M, N), -9, dtype=_TDT[dtype], device="cuda")
        vla.vla_ternary_linear(packed, beta, x, M, N, K, ref, dtype, vla.VLA_PATH_AUTO, None, None, ws, nb)
        vla.vla_ternary_linear_static(packed, beta, x, M, N, K, got, dtype, vla.VLA_PATH_AUTO)
        torch.cuda.synchronize()
        assert np.array_equal(_raw(got), _raw(ref)), "call %d differs from the workspace path" % call
        if dtype == 0:                                               # and within the fp32 tolerance of test_gpu_parity.py
            a, b = got.double().cpu().numpy(), ref.double().cpu().numpy()
            assert np.all(np.abs(a - b) <= 1e-6 * np.abs(b))


@pytest.mark.gpu
def test_static_entry_point_rejects_oversize_on_the_device(vla):
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    K, N = 8192, 128
    M = vla.VLA_STATIC_MAX_MK // K + 1
    x = torch.zeros((M, K), dtype=torch.bfloat16, device="cuda")
    w = torch.zeros((N, K), dtype=torch.int8, device="cuda")
    packed = vla.pack_weights(w)
    beta = torch.ones(1, dtype=torch.float32, device="cuda")
    out = torch.empty((M, N), dtype=torch.float32, device="cuda")
    with pytest.raises(vla.VlaError) as e:
        vla.vla_ternary_linear_static(packed, beta, x, M, N, K, out, 0)
    assert e.value.status == vla.VLA_ERR_WORKSPACE
    vla.vla_ternary_linear_static(packed, beta, x[:M - 1], M - 1, N, K, out[:M - 1], 0)       # exactly at the limit: fine
    torch.cuda.synchronize()
    assert bool((out[:M - 1] == 0).all())
