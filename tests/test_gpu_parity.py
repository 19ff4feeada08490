"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI, against the CPU oracle, element by
element on the same seeded inputs.  Bars (BASELINE.json north_star): int8 activations, fp32 alpha and
int32 accumulators bit-exact; fp32 outputs within 1e-6 relative of the fp64 reference; bf16 outputs
within 1 bf16 ulp of RNE(fp64 reference).  With the canonical operation order of DESIGN.md (readings
R1, R6) the fp32 and bf16 outputs are also bit-identical to the oracle's, which is asserted too.
"""
import ctypes
import os

import numpy as np
import pytest
import torch

from paper_2606_08094_b200 import synth

pytestmark = pytest.mark.gpu

REL_TOL_F32 = 1e-6          # north_star: "fp32 outputs must agree within 1e-6 relative"


@pytest.fixture(scope="module")
def vla():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    from paper_2606_08094_b200 import binding
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def dev_bf16(bits_u16):
    return torch.from_numpy(np.ascontiguousarray(bits_u16).view(np.int16)).cuda().view(torch.bfloat16)


def bf16_bits_of(t):
    return t.view(torch.int16).cpu().numpy().view(np.uint16)


def bf16_ulp_distance(a_bits, b_bits):
    """distance in units of bf16 ulps between two arrays of finite bf16 bit patterns (monotone integer map)"""
    def key(b):
        b = b.astype(np.int32)
        return np.where(b & 0x8000, -(b & 0x7FFF), b & 0x7FFF)
    return np.abs(key(a_bits) - key(b_bits))


def run_gemm(vla, packed, beta, xq, xs, M, N, K, out_dtype, path):
    out = vla.empty_out(M, N, out_dtype)
    ws_bytes = vla.vla_ternary_workspace_bytes(M, N, K, path)
    ws = torch.empty(max(ws_bytes, 16), dtype=torch.uint8, device="cuda")
    vla.vla_ternary_gemm(packed, beta, xq, xs, M, N, K, out, out_dtype, path, ws, ws_bytes)
    torch.cuda.synchronize()
    return out


def check_outputs(vla, oracle, packed, w, beta, x_bits, M, N, K, path):
    """act_quant + gemm (all three output dtypes) on `path` vs the oracle."""
    ref = oracle.ternary_linear(x_bits, w, beta)
    x = dev_bf16(x_bits)
    xq = torch.empty((M, K), dtype=torch.int8, device="cuda")
    xs = torch.empty((M,), dtype=torch.float32, device="cuda")
    vla.vla_act_quant(x, M, K, xq, xs)
    torch.cuda.synchronize()
    assert np.array_equal(xq.cpu().numpy(), ref["a"]), "int8 activations differ"
    assert np.array_equal(xs.cpu().numpy().view(np.uint32), ref["alpha"].view(np.uint32)), "alpha differs"
    beta_d = dev(np.array([beta], np.float32))

    acc = run_gemm(vla, packed, beta_d, xq, xs, M, N, K, vla.VLA_I32, path).cpu().numpy()
    bad = np.argwhere(acc != ref["acc"])
    assert bad.size == 0, "int32 accumulators differ at %d places, first %s: got %d want %d" % (
        len(bad), bad[0], acc[tuple(bad[0])], ref["acc"][tuple(bad[0])])

    y = run_gemm(vla, packed, beta_d, xq, xs, M, N, K, vla.VLA_F32, path).cpu().numpy()
    y64 = ref["y64"]
    err = np.abs(y.astype(np.float64) - y64)
    assert np.all(err <= REL_TOL_F32 * np.abs(y64)), "fp32 output outside 1e-6 relative"
    assert np.all(y[ref["acc"] == 0] == 0.0)
    assert np.array_equal(y.view(np.uint32), ref["y32"].view(np.uint32)), "fp32 output not bit-identical"

    yb = bf16_bits_of(run_gemm(vla, packed, beta_d, xq, xs, M, N, K, vla.VLA_BF16, path))
    want = oracle.f32_to_bf16(y64.astype(np.float32))
    assert bf16_ulp_distance(yb, want).max() <= 1, "bf16 output more than 1 ulp from RNE(reference)"
    assert np.array_equal(yb, ref["ybf16"]), "bf16 output not bit-identical"
    return ref


def paths_for(vla, M):
    p = [vla.VLA_PATH_LARGE]
    if M <= 16:
        p.append(vla.VLA_PATH_SMALL_ALU)
    if M <= 32:
        p.append(vla.VLA_PATH_SMALL_TC)
    return p


# ---------------------------------------------------------------- packer
@pytest.mark.parametrize("N,K", [(128, 128), (256, 256), (384, 640), (2560, 2560), (640, 2560)])
def test_pack_unpack_round_trip(vla, N, K):
    w = synth.ternary_weights(N, K, 0.35, 42 + N + K)
    wd = dev(w)
    packed = vla.pack_weights(wd)
    assert packed.numel() == N * K // 4
    back = torch.full((N, K), 99, dtype=torch.int8, device="cuda")
    vla.vla_ternary_unpack(packed, N, K, back)
    torch.cuda.synchronize()
    assert torch.equal(back, wd)


def test_pack_rejects_non_ternary(vla):
    w = synth.ternary_weights(128, 256, 0.3, 1)
    for bad in (2, -2, 127, -128):
        w2 = w.copy()
        w2[77, 133] = bad
        with pytest.raises(vla.VlaError) as e:
            vla.pack_weights(dev(w2))
        assert e.value.status == vla.VLA_ERR_VALUE


# ---------------------------------------------------------------- quantiser
@pytest.mark.parametrize("M,K", [(1, 128), (8, 256), (16, 2560), (13, 6912), (544, 2560), (37, 8192), (3, 16384)])
def test_act_quant_bit_exact(vla, oracle, M, K):
    x_bits = synth.activations(M, K, 900 + M + K, outlier_frac=0.01)
    a_ref, al_ref = oracle.act_quant(x_bits)
    xq = torch.empty((M, K), dtype=torch.int8, device="cuda")
    xs = torch.empty((M,), dtype=torch.float32, device="cuda")
    vla.vla_act_quant(dev_bf16(x_bits), M, K, xq, xs)
    torch.cuda.synchronize()
    assert np.array_equal(xq.cpu().numpy(), a_ref)
    assert np.array_equal(xs.cpu().numpy().view(np.uint32), al_ref.view(np.uint32))


def test_act_quant_special_rows(vla, oracle):
    """ties (0.8125, 0.40625 -> 127, 63 under true division), all-zero row, tiny row, heavy tails, negatives."""
    K = 128
    rows = np.zeros((6, K), np.float32)
    rows[0, :2] = [0.8125, 0.40625]
    rows[1, :4] = [1.0, -0.5, 0.25, 2.0]
    rows[3, :3] = [3e-6, -1e-6, 2e-6]
    rows[4] = np.random.default_rng(5).standard_t(3.0, K).astype(np.float32) * 50
    rows[5] = -np.abs(np.random.default_rng(6).standard_normal(K).astype(np.float32))
    x_bits = synth._f32_to_bf16_bits(rows)
    a_ref, al_ref = oracle.act_quant(x_bits)
    assert a_ref[0, :2].tolist() == [127, 63]
    xq = torch.empty((6, K), dtype=torch.int8, device="cuda")
    xs = torch.empty((6,), dtype=torch.float32, device="cuda")
    vla.vla_act_quant(dev_bf16(x_bits), 6, K, xq, xs)
    torch.cuda.synchronize()
    assert np.array_equal(xq.cpu().numpy(), a_ref)
    assert np.array_equal(xs.cpu().numpy().view(np.uint32), al_ref.view(np.uint32))
    assert xq[2].abs().max().item() == 0


# ---------------------------------------------------------------- GEMM paths
def test_config0_smoke_all_paths(vla, oracle):
    c = synth.config0()
    packed = vla.pack_weights(dev(c["w"]))
    for path in paths_for(vla, c["M"]) + [vla.VLA_PATH_AUTO]:
        check_outputs(vla, oracle, packed, c["w"], c["beta"], c["x"], c["M"], c["N"], c["K"], path)


@pytest.mark.parametrize("M", [1, 2, 3, 5, 8, 11, 16, 17, 32, 33, 100, 128, 129, 300])
@pytest.mark.parametrize("N,K", [(128, 128), (384, 640), (640, 1152)])
def test_small_shapes_ragged_m(vla, oracle, M, N, K):
    """several tiles and ragged tails in every dimension the kernels tile (M, N/128, K/128)"""
    w = synth.ternary_weights(N, K, 0.33, 7 * N + K)
    x = synth.activations(M, K, 31 * M + K, dist="student_t3")
    packed = vla.pack_weights(dev(w))
    for path in paths_for(vla, M):
        check_outputs(vla, oracle, packed, w, np.float32(0.037), x, M, N, K, path)


@pytest.mark.parametrize("shape_idx", [0, 1, 2, 3])
@pytest.mark.parametrize("M", [1, 8, 16])
def test_config1_decode_points(vla, oracle, shape_idx, M):
    c = synth.config1_point(shape_idx, M)
    packed = vla.pack_weights(dev(c["w"]))
    for path in paths_for(vla, M) + [vla.VLA_PATH_AUTO]:
        check_outputs(vla, oracle, packed, c["w"], c["beta"], c["x"], M, c["N"], c["K"], path)


@pytest.mark.parametrize("shape_idx", [0, 1, 2, 3])
def test_config2_prefill_points_fused_linear(vla, oracle, shape_idx):
    """configs[2]: M=544 with the quant fused into the call (vla_ternary_linear), fp32 output."""
    c = synth.config2_point(shape_idx)
    M, N, K = c["M"], c["N"], c["K"]
    packed = vla.pack_weights(dev(c["w"]))
    ref = check_outputs(vla, oracle, packed, c["w"], c["beta"], c["x"], M, N, K, vla.VLA_PATH_LARGE)
    out = vla.empty_out(M, N, vla.VLA_F32)
    xq = torch.empty((M, K), dtype=torch.int8, device="cuda")
    xs = torch.empty((M,), dtype=torch.float32, device="cuda")
    ws_bytes = vla.vla_ternary_workspace_bytes(M, N, K)
    ws = torch.empty(ws_bytes, dtype=torch.uint8, device="cuda")
    beta_d = dev(np.array([c["beta"]], np.float32))
    vla.vla_ternary_linear(packed, beta_d, dev_bf16(c["x"]), M, N, K, out, vla.VLA_F32, vla.VLA_PATH_AUTO,
                           xq, xs, ws, ws_bytes)
    torch.cuda.synchronize()
    assert np.array_equal(xq.cpu().numpy(), ref["a"])
    assert np.array_equal(out.cpu().numpy().view(np.uint32), ref["y32"].view(np.uint32))
    # same call with the quantised activations kept in the workspace
    out2 = vla.empty_out(M, N, vla.VLA_F32)
    vla.vla_ternary_linear(packed, beta_d, dev_bf16(c["x"]), M, N, K, out2, vla.VLA_F32, vla.VLA_PATH_AUTO,
                           None, None, ws, ws_bytes)
    torch.cuda.synchronize()
    assert torch.equal(out, out2)


def test_sweep_shape_8192_sampled(vla, oracle):
    """configs[4] largest shape at M=512: full int32 parity (the oracle needs ~34 G MACs: seconds on 8 cores)."""
    c = synth.config4_point(512, 3, 1, 1)
    M, N, K = 512, c["N"], c["K"]
    packed = vla.pack_weights(dev(c["w"]))
    a_ref, al_ref = oracle.act_quant(c["x"])
    xq = torch.empty((M, K), dtype=torch.int8, device="cuda")
    xs = torch.empty((M,), dtype=torch.float32, device="cuda")
    vla.vla_act_quant(dev_bf16(c["x"]), M, K, xq, xs)
    assert np.array_equal(xq.cpu().numpy(), a_ref)
    beta_d = dev(np.array([c["beta"]], np.float32))
    acc = run_gemm(vla, packed, beta_d, xq, xs, M, N, K, vla.VLA_I32, vla.VLA_PATH_LARGE).cpu().numpy()
    # sampled rows of the output (every 37th token), each a full row of N dot products
    rows = np.arange(0, M, 37)
    ref = oracle.contract(a_ref[rows], c["w"])
    assert np.array_equal(acc[rows], ref)


# ---------------------------------------------------------------- invariants through the CUDA path
@pytest.mark.parametrize("M", [8, 64])
def test_unit_vector_activations_return_w_columns(vla, M):
    """x_m = c * e_j  ->  acc_mn = 127 * w_nj exactly: catches any K permutation in the packed layout."""
    N, K = 256, 512
    w = synth.ternary_weights(N, K, 0.3, 77)
    packed = vla.pack_weights(dev(w))
    rng = np.random.default_rng(3)
    js = rng.choice(K, size=M, replace=False)
    x = np.zeros((M, K), np.float32)
    x[np.arange(M), js] = rng.uniform(0.5, 3.0, M).astype(np.float32)
    xq = torch.empty((M, K), dtype=torch.int8, device="cuda")
    xs = torch.empty((M,), dtype=torch.float32, device="cuda")
    vla.vla_act_quant(dev_bf16(synth._f32_to_bf16_bits(x)), M, K, xq, xs)
    beta_d = dev(np.array([1.0], np.float32))
    for path in paths_for(vla, M):
        acc = run_gemm(vla, packed, beta_d, xq, xs, M, N, K, vla.VLA_I32, path).cpu().numpy()
        assert np.array_equal(acc, 127 * w[:, js].T.astype(np.int32))


def test_all_ones_weights_return_row_sums(vla):
    M, N, K = 16, 256, 640
    for val in (1, -1, 0):
        w = np.full((N, K), val, np.int8)
        packed = vla.pack_weights(dev(w))
        x_bits = synth.activations(M, K, 11)
        xq = torch.empty((M, K), dtype=torch.int8, device="cuda")
        xs = torch.empty((M,), dtype=torch.float32, device="cuda")
        vla.vla_act_quant(dev_bf16(x_bits), M, K, xq, xs)
        rows = xq.cpu().numpy().astype(np.int64).sum(axis=1) * val
        beta_d = dev(np.array([1.0], np.float32))
        for path in paths_for(vla, M):
            acc = run_gemm(vla, packed, beta_d, xq, xs, M, N, K, vla.VLA_I32, path).cpu().numpy()
            assert np.array_equal(acc, np.repeat(rows[:, None], N, axis=1))


def test_extreme_accumulators(vla):
    """|acc| reaches 127*K: all activations saturate at +-127 and W = sign pattern (K = 8192, the sweep's max)."""
    M, N, K = 4, 128, 8192
    x = np.ones((M, K), np.float32)
    x[1] = -1.0
    x[2, ::2] = -1.0
    w = np.ones((N, K), np.int8)
    w[1::2] = -1
    packed = vla.pack_weights(dev(w))
    xq = torch.empty((M, K), dtype=torch.int8, device="cuda")
    xs = torch.empty((M,), dtype=torch.float32, device="cuda")
    vla.vla_act_quant(dev_bf16(synth._f32_to_bf16_bits(x)), M, K, xq, xs)
    want = xq.cpu().numpy().astype(np.int64) @ w.T.astype(np.int64)
    assert np.abs(want).max() == 127 * K
    beta_d = dev(np.array([1.0], np.float32))
    for path in paths_for(vla, M):
        acc = run_gemm(vla, packed, beta_d, xq, xs, M, N, K, vla.VLA_I32, path).cpu().numpy()
        assert np.array_equal(acc, want)


# ---------------------------------------------------------------- host-buffer entry point + errors on a GPU
def test_linear_host_round_trip(vla, oracle):
    c = synth.config1_point(1, 8)
    M, N, K = c["M"], c["N"], c["K"]
    packed = vla.pack_weights(dev(c["w"]))
    ref = oracle.ternary_linear(c["x"], c["w"], c["beta"])
    xh = torch.from_numpy(c["x"].view(np.int16)).view(torch.bfloat16).pin_memory()
    oh = torch.empty((M, N), dtype=torch.bfloat16).pin_memory()
    nb = vla.vla_ternary_host_workspace_bytes(M, N, K, vla.VLA_BF16)
    ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
    beta_d = dev(np.array([c["beta"]], np.float32))
    vla.vla_ternary_linear_host(packed, beta_d, xh, M, N, K, oh, vla.VLA_BF16, vla.VLA_PATH_AUTO, ws, nb)
    assert np.array_equal(oh.view(torch.int16).numpy().view(np.uint16), ref["ybf16"])


def test_errors_on_device(vla):
    w = dev(synth.ternary_weights(128, 128, 0.3, 1))
    packed = vla.pack_weights(w)
    out = vla.empty_out(8, 128, vla.VLA_F32)
    xq = torch.zeros((8, 128), dtype=torch.int8, device="cuda")
    xs = torch.ones((8,), dtype=torch.float32, device="cuda")
    beta = torch.ones((1,), dtype=torch.float32, device="cuda")
    with pytest.raises(vla.VlaError) as e:
        vla.vla_ternary_gemm(packed, beta, xq, xs, 64, 128, 128, out, vla.VLA_F32, vla.VLA_PATH_SMALL_ALU)
    assert e.value.status == vla.VLA_ERR_SHAPE
    with pytest.raises(vla.VlaError) as e:
        vla.vla_ternary_gemm(packed, beta, xq.data_ptr() + 1, xs, 8, 128, 128, out, vla.VLA_F32)
    assert e.value.status == vla.VLA_ERR_ALIGN
    launches = vla.vla_launch_count()
    vla.vla_ternary_gemm(packed, beta, xq, xs, 8, 128, 128, out, vla.VLA_F32)
    torch.cuda.synchronize()
    assert vla.vla_launch_count() > launches
    assert torch.all(out == 0)


def test_library_is_the_loaded_native_code(vla):
    """the in-tree .so is what the process mapped (no silent eager fallback exists)"""
    maps = open("/proc/self/maps").read()
    assert os.path.basename(vla.LIB_PATH) in maps


# ---------------------------------------------------------------- full-size shapes, sampled output channels
@pytest.mark.parametrize("M,K,N", [(4096, 8192, 8192), (1024, 6912, 2560), (2048, 2560, 6912)])
def test_full_size_large_m_sampled_channels(vla, oracle, M, K, N):
    """BASELINE.json configs[4] sizes in the launch configuration bench.py --workload sweep times (fused quant, fp32
    out, VLA_PATH_AUTO).  The oracle cannot do 2.7e11 MACs in seconds, so it computes 64 sampled output channels
    (all M tokens, all of K) one by one; every activation row is checked in full."""
    rng = np.random.Generator(np.random.PCG64(M + K + N))
    w = synth.ternary_weights(N, K, 0.33, 77 + N)
    x_bits = synth.activations(M, K, 78 + K, dist="student_t3")
    beta = np.float32(0.05)
    cols = np.sort(rng.choice(N, size=64, replace=False))
    ref = oracle.ternary_linear(x_bits, np.ascontiguousarray(w[cols]), beta)
    packed = vla.pack_weights(dev(w))
    x = dev_bf16(x_bits)
    xq = torch.empty((M, K), dtype=torch.int8, device="cuda")
    xs = torch.empty((M,), dtype=torch.float32, device="cuda")
    nb = vla.vla_ternary_workspace_bytes(M, N, K)
    ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
    beta_d = dev(np.array([beta], np.float32))
    for dtype, key in ((vla.VLA_I32, "acc"), (vla.VLA_F32, "y32")):
        out = vla.empty_out(M, N, dtype)
        vla.vla_ternary_linear(packed, beta_d, x, M, N, K, out, dtype, vla.VLA_PATH_AUTO, xq, xs, ws, nb)
        torch.cuda.synchronize()
        got = out[:, torch.from_numpy(cols).cuda()].cpu().numpy()
        if key == "acc":
            assert np.array_equal(got, ref["acc"])
        else:
            assert np.array_equal(got.view(np.uint32), ref["y32"].view(np.uint32))
            assert np.all(np.abs(got.astype(np.float64) - ref["y64"]) <= REL_TOL_F32 * np.abs(ref["y64"]))
    assert np.array_equal(xq.cpu().numpy(), ref["a"])
    assert np.array_equal(xs.cpu().numpy().view(np.uint32), ref["alpha"].view(np.uint32))


@pytest.mark.parametrize("M", [17, 32])
@pytest.mark.parametrize("N,K,want", [(2560, 2560, "large"), (640, 2560, "small_tc"), (2560, 6912, "small_tc")])
def test_auto_path_between_16_and_32_tokens(vla, oracle, M, N, K, want):
    """Row a6: for 16 < M <= 32 VLA_PATH_AUTO picks by (N,K); whichever kernel it picks, the call matches
    the oracle bit for bit."""
    expect = vla.VLA_PATH_LARGE if want == "large" else vla.VLA_PATH_SMALL_TC
    assert vla.vla_ternary_auto_path(M, N, K) == expect
    w = synth.ternary_weights(N, K, 0.35, 77 + N + K)
    x = synth.activations(M, K, 1700 + M + K, outlier_frac=0.01)
    packed = vla.pack_weights(dev(w))
    check_outputs(vla, oracle, packed, w, np.float32(0.021), x, M, N, K, vla.VLA_PATH_AUTO)


def test_grouped_auto_at_24_tokens_matches_per_linear_calls(vla, oracle):
    """q|k|v at M = 24 through VLA_PATH_AUTO: the group's total N decides the kernel; outputs are the oracle's."""
    M, K = 24, 2560
    x_bits = synth.activations(M, K, 2424, outlier_frac=0.01)
    xq = torch.empty((M, K), dtype=torch.int8, device="cuda")
    xs = torch.empty((M,), dtype=torch.float32, device="cuda")
    vla.vla_act_quant(dev_bf16(x_bits), M, K, xq, xs)
    lins, keep = [], []
    for i, (N, beta) in enumerate([(2560, 0.05), (640, 0.013), (640, 0.5)]):
        w = synth.ternary_weights(N, K, 0.35, 950 + i)
        packed = vla.pack_weights(dev(w))
        beta_d = dev(np.array([beta], np.float32))
        out = vla.empty_out(M, N, vla.VLA_F32)
        keep.append((w, packed, beta_d, out, np.float32(beta)))
        lins.append(dict(packed=packed, w_scale=beta_d, out=out, N=N, out_dtype=vla.VLA_F32))
    vla.vla_ternary_gemm_grouped(lins, xq, xs, M, K, vla.VLA_PATH_AUTO)
    torch.cuda.synchronize()
    for (w, packed, beta_d, out, beta) in keep:
        ref = oracle.ternary_linear(x_bits, w, beta)
        assert np.array_equal(out.cpu().numpy().view(np.uint32), ref["y32"].view(np.uint32))


def test_grouped_large_gemm_per_group_scales(vla, oracle):
    """q|k|v-style group: three linears with their own beta and output type share one quantised activation matrix and
    run as ONE tcgen05 launch (Eq. 4's per-output-group scales); ragged M, every linear vs the oracle."""
    M, K = 200, 640
    x_bits = synth.activations(M, K, 4242, outlier_frac=0.01)
    x = dev_bf16(x_bits)
    xq = torch.empty((M, K), dtype=torch.int8, device="cuda")
    xs = torch.empty((M,), dtype=torch.float32, device="cuda")
    vla.vla_act_quant(x, M, K, xq, xs)
    specs = [(256, vla.VLA_BF16, 0.05), (128, vla.VLA_F32, 0.013), (384, vla.VLA_I32, 0.5)]
    lins, keep = [], []
    for i, (N, dt, beta) in enumerate(specs):
        w = synth.ternary_weights(N, K, 0.35, 900 + i)
        packed = vla.pack_weights(dev(w))
        beta_d = dev(np.array([beta], np.float32))
        out = vla.empty_out(M, N, dt)
        keep.append((w, packed, beta_d, out, np.float32(beta), dt))
        lins.append(dict(packed=packed, w_scale=beta_d, out=out, N=N, out_dtype=dt))
    vla.vla_ternary_gemm_grouped(lins, xq, xs, M, K, vla.VLA_PATH_LARGE)
    torch.cuda.synchronize()
    for (w, packed, beta_d, out, beta, dt) in keep:
        ref = oracle.ternary_linear(x_bits, w, beta)
        if dt == vla.VLA_I32:
            assert np.array_equal(out.cpu().numpy(), ref["acc"])
        elif dt == vla.VLA_F32:
            assert np.array_equal(out.cpu().numpy().view(np.uint32), ref["y32"].view(np.uint32))
        else:
            assert np.array_equal(bf16_bits_of(out), ref["ybf16"])


def test_grouped_full_size_ragged_mixed_dtypes(vla, oracle):
    """The grouped tcgen05 launch at model size with a ragged token count (M = 545: one token past the prefill's 544) and
    mixed output types: gate|up|k-like group, K = 2560, N = 6912 | 6912 | 640 (113 channel tiles over several waves, tiles
    of three linears in one walk).  Rows are sampled for the oracle (its int32 contraction is exact per row)."""
    M, K = 545, 2560
    x_bits = synth.activations(M, K, 4343, outlier_frac=0.01)
    x = dev_bf16(x_bits)
    xq = torch.empty((M, K), dtype=torch.int8, device="cuda")
    xs = torch.empty((M,), dtype=torch.float32, device="cuda")
    vla.vla_act_quant(x, M, K, xq, xs)
    specs = [(6912, vla.VLA_BF16, 0.021), (6912, vla.VLA_F32, 0.3), (640, vla.VLA_I32, 0.07)]
    lins, keep = [], []
    for i, (N, dt, beta) in enumerate(specs):
        w = synth.ternary_weights(N, K, 0.35, 950 + i)
        beta_d = dev(np.array([beta], np.float32))
        out = vla.empty_out(M, N, dt)
        keep.append((w, beta_d, out, np.float32(beta), dt))
        lins.append(dict(packed=vla.pack_weights(dev(w)), w_scale=beta_d, out=out, N=N, out_dtype=dt))
    vla.vla_ternary_gemm_grouped(lins, xq, xs, M, K, vla.VLA_PATH_AUTO)
    torch.cuda.synchronize()
    rows = np.array([0, 1, 95, 96, 127, 128, 255, 256, 300, 511, 512, 543, 544])
    for (w, beta_d, out, beta, dt) in keep:
        ref = oracle.ternary_linear(np.ascontiguousarray(x_bits[rows]), w, beta)
        got = out[torch.from_numpy(rows).cuda()]
        if dt == vla.VLA_I32:
            assert np.array_equal(got.cpu().numpy(), ref["acc"])
        elif dt == vla.VLA_F32:
            assert np.array_equal(got.cpu().numpy().view(np.uint32), ref["y32"].view(np.uint32))
        else:
            assert np.array_equal(bf16_bits_of(got.contiguous()), ref["ybf16"])


def test_grouped_equal_groups_vs_oracle_group_vector(vla, oracle):
    """Eq. 4's beta_g(n) in the oracle's own form: three equal output groups with a [G=3] scale vector (the branch pinned
    by test_ternary_linear_bf16_with_three_output_groups_vs_exact) against ONE grouped launch of three linears."""
    M, K, Ng = 77, 1280, 256
    x_bits = synth.activations(M, K, 4444, outlier_frac=0.01)
    xq = torch.empty((M, K), dtype=torch.int8, device="cuda")
    xs = torch.empty((M,), dtype=torch.float32, device="cuda")
    vla.vla_act_quant(dev_bf16(x_bits), M, K, xq, xs)
    w = synth.ternary_weights(3 * Ng, K, 0.35, 960)
    betas = np.array([0.013, 0.4, 0.077], np.float32)
    outs, lins, keep = [], [], []
    for g in range(3):
        out = vla.empty_out(M, Ng, vla.VLA_BF16)
        bd = dev(betas[g:g + 1])
        keep.append(bd)
        outs.append(out)
        lins.append(dict(packed=vla.pack_weights(dev(w[g * Ng:(g + 1) * Ng])), w_scale=bd, out=out, N=Ng, out_dtype=vla.VLA_BF16))
    vla.vla_ternary_gemm_grouped(lins, xq, xs, M, K, vla.VLA_PATH_LARGE)
    torch.cuda.synchronize()
    ref = oracle.ternary_linear(x_bits, w, betas)
    for g in range(3):
        assert np.array_equal(bf16_bits_of(outs[g]), ref["ybf16"][:, g * Ng:(g + 1) * Ng]), "group %d" % g


def test_longest_supported_k_saturating(vla):
    """K = 65536, the largest K the ABI accepts: saturated activations (+-127) against sign-pattern weights, |acc| =
    127 * 65536 (the decode's factor 64 leaves 64 * 127 * K < 2^31), on every path that takes this M."""
    M, N, K = 4, 128, 65536
    x = np.ones((M, K), np.float32)
    x[1] = -1.0
    x[2, ::2] = -1.0
    x[3, ::3] = 0.5
    w = np.ones((N, K), np.int8)
    w[1::2] = -1
    w[5, ::7] = 0
    packed = vla.pack_weights(dev(w))
    xq = torch.empty((M, K), dtype=torch.int8, device="cuda")
    xs = torch.empty((M,), dtype=torch.float32, device="cuda")
    vla.vla_act_quant(dev_bf16(synth._f32_to_bf16_bits(x)), M, K, xq, xs)
    want = xq.cpu().numpy().astype(np.int64) @ w.T.astype(np.int64)
    assert np.abs(want).max() == 127 * K
    beta_d = dev(np.array([1.0], np.float32))
    for path in paths_for(vla, M):
        acc = run_gemm(vla, packed, beta_d, xq, xs, M, N, K, vla.VLA_I32, path).cpu().numpy()
        assert np.array_equal(acc, want), "path %d" % path


def test_forced_path_token_limits(vla):
    """include/vla_ternary.h: VLA_PATH_SMALL_ALU takes M <= 16, VLA_PATH_SMALL_TC M <= 32; one more token is VLA_ERR_SHAPE."""
    K, N = 256, 128
    packed = vla.pack_weights(dev(synth.ternary_weights(N, K, 0.3, 3)))
    beta_d = dev(np.array([0.05], np.float32))
    for path, mmax in ((vla.VLA_PATH_SMALL_ALU, 16), (vla.VLA_PATH_SMALL_TC, 32)):
        for M, ok in ((mmax, True), (mmax + 1, False)):
            xq = torch.zeros((M, K), dtype=torch.int8, device="cuda")
            xs = torch.ones((M,), dtype=torch.float32, device="cuda")
            out = vla.empty_out(M, N, vla.VLA_F32)
            if ok:
                vla.vla_ternary_gemm(packed, beta_d, xq, xs, M, N, K, out, vla.VLA_F32, path, None, 0)
            else:
                with pytest.raises(vla.VlaError) as e:
                    vla.vla_ternary_gemm(packed, beta_d, xq, xs, M, N, K, out, vla.VLA_F32, path, None, 0)
                assert e.value.status == vla.VLA_ERR_SHAPE
    torch.cuda.synchronize()


@pytest.mark.parametrize("M,path_name", [(7, "small_tc"), (7, "small_alu"), (37, "large"), (200, "large")])
def test_guard_bands_single_calls(vla, oracle, M, path_name):
    """Sentinel bytes around xq, alpha and the output survive act_quant + GEMM on every path (ragged M)."""
    path = {"small_tc": vla.VLA_PATH_SMALL_TC, "small_alu": vla.VLA_PATH_SMALL_ALU, "large": vla.VLA_PATH_LARGE}[path_name]
    K, N = 384, 256
    def guarded(shape, dtype):
        n = int(np.prod(shape)) * torch.empty((), dtype=dtype).element_size()
        raw = torch.full((n + 8192,), 0xA5, dtype=torch.uint8, device="cuda")
        return raw, raw[4096:4096 + n].view(dtype).view(*shape)
    x_bits = synth.activations(M, K, 55 + M)
    w = synth.ternary_weights(N, K, 0.35, 56)
    beta = np.float32(0.07)
    rq, xq = guarded((M, K), torch.int8)
    rs, xs = guarded((M,), torch.float32)
    ro, out = guarded((M, N), torch.float32)
    packed = vla.pack_weights(dev(w))
    vla.vla_act_quant(dev_bf16(x_bits), M, K, xq, xs)
    vla.vla_ternary_gemm(packed, dev(np.array([beta], np.float32)), xq, xs, M, N, K, out, vla.VLA_F32, path, None, 0)
    torch.cuda.synchronize()
    ref = oracle.ternary_linear(x_bits, w, beta)
    assert np.array_equal(out.cpu().numpy().view(np.uint32), ref["y32"].view(np.uint32))
    for raw in (rq, rs, ro):
        r = raw.cpu().numpy()
        assert (r[:4096] == 0xA5).all() and (r[-4096:] == 0xA5).all(), "a kernel wrote outside its buffer"
