"""Host-side validation of the program API (no GPU needed): vla_program_bytes / vla_program_build answer from the
host before any launch, and there is no CPU fallback behind vla_program_run."""
import pytest


@pytest.fixture(scope="module")
def vla():
    from paper_2606_08094_b200 import binding
    return binding


FAKE = 0x10000   # 256-byte aligned non-NULL "pointer"; never dereferenced because validation comes first


def stage(M=8, K=2560, N=2560, depends=0, n=1, dtype=1):
    return dict(x=FAKE, M=M, K=K, depends=depends,
                linears=[dict(packed=FAKE, w_scale=FAKE, out=FAKE, N=N, out_dtype=dtype) for _ in range(n)])


def test_program_bytes_counts_tables_counters_and_cooperative_scratch(vla):
    """the device buffer holds the descriptor tables, the counters and, for stages quantised cooperatively (more than
    1440 sixteen-element tasks), the int8 fragments + alpha; small stages are quantised in shared memory and add nothing"""
    small = vla.vla_program_bytes([stage(M=1)])                      # 160 tasks: local
    assert small % 256 == 0 and 512 <= small < 4096
    assert vla.vla_program_bytes([stage()]) == small                 # M=8, K=2560: 1280 tasks, still local
    one = vla.vla_program_bytes([stage(M=16)])                       # 2560 tasks: cooperative, 16*2560 B of fragments
    assert small + 16 * 2560 <= one < small + 16 * 2560 + 1024
    two = vla.vla_program_bytes([stage(M=16), stage(M=8, K=6912, depends=1)])
    assert one + 8 * 6912 <= two < one + 8 * 6912 + 1024


@pytest.mark.parametrize("bad", [dict(M=0), dict(M=32769), dict(M=64, n=9), dict(M=64, K=8192 + 128), dict(K=100), dict(K=8192 + 128), dict(N=100), dict(N=0),
                                 dict(depends=2), dict(n=0), dict(n=17), dict(dtype=3)])
def test_invalid_stage_gives_zero_bytes(vla, bad):
    assert vla.vla_program_bytes([stage(**bad)]) == 0


def test_one_kind_per_program_and_large_program_bytes(vla):
    """stages with M > 16 tokens form a LARGE program (persistent tcgen05 kernel): not mixable with small stages; its
    buffer holds the stage table (tensor map + group per stage), the counters and eight {int8 [M,K], alpha [M]} scratch sets"""
    assert vla.vla_program_bytes([stage(M=8), stage(M=64)]) == 0
    assert vla.vla_program_bytes([stage(M=64), stage(M=16)]) == 0
    one = vla.vla_program_bytes([stage(M=544)])
    assert one % 256 == 0 and 8 * 544 * 2560 <= one < 8 * 544 * 2560 + 65536
    two = vla.vla_program_bytes([stage(M=544), stage(M=100, K=6912, depends=1, n=2)])
    assert 8 * 544 * 2560 <= two < 8 * 544 * 2560 + 65536 and two > one


def test_descriptor_capacity_is_enforced(vla):
    # 30 layers x 4 stages with 7 linears fit (BASELINE.json configs[3]); ten times that does not
    layer = [stage(n=3), stage(depends=1), stage(n=2, depends=1), stage(K=6912, depends=1)]
    assert vla.vla_program_bytes(layer * 30) > 0
    assert vla.vla_program_bytes(layer * 300) == 0


def test_build_and_run_validate_on_the_host(vla):
    arr, _keep = vla._marshal_stages([stage()])
    L = vla._lib
    assert L.vla_program_build(arr, 1, None, 1 << 20, None) == vla.VLA_ERR_NULL
    assert L.vla_program_build(arr, 1, FAKE + 16, 1 << 20, None) == vla.VLA_ERR_ALIGN
    assert L.vla_program_build(arr, 1, FAKE, 16, None) == vla.VLA_ERR_WORKSPACE
    assert L.vla_program_build(None, 1, FAKE, 1 << 20, None) == vla.VLA_ERR_NULL
    assert L.vla_program_run(None, None) == vla.VLA_ERR_NULL
    assert L.vla_program_run(FAKE, None) == vla.VLA_ERR_VALUE          # never compiled
    assert L.vla_program_release(FAKE) == vla.VLA_ERR_VALUE
    assert L.vla_program_run_host(FAKE, None, 1, None, 0, None) == vla.VLA_ERR_NULL
    assert L.vla_program_run_host_async(FAKE, None, 1, None, 0, None) == vla.VLA_ERR_NULL
    assert L.vla_program_run_host_async(FAKE, None, 0, None, 0, None) == vla.VLA_ERR_VALUE     # never compiled


def test_no_gpu_means_arch_error(vla):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    arr, _keep = vla._marshal_stages([stage()])
    assert vla._lib.vla_program_build(arr, 1, FAKE, 1 << 20, None) == vla.VLA_ERR_ARCH
