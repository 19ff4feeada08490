"""GPU parity (-m gpu) of the cached-conditioning cross-attention (vla_cached_attention, Eq. 2 of the paper, PAPER.md
lines 48-54) against oracle/attention.py (float64, the definition written out).

Tolerance: the kernel computes the scores and the weighted sums in fp32 from exact bf16 products, keeps
the probabilities to 2^-17 relative (hi + lo bf16 split) and uses exp2f on (s - max) * log2(e)/sqrt(d_k).  Error sources
per output: score rounding 2^-24 * sum|q k| * c  -> relative 1e-6 on each probability for |s| <= 30; exp2f 2 ulp; the P
split 2^-17; fp32 accumulation over Mc keys 2^-24 * Mc.  Together < 2e-5 relative to sum_j p_j |v_j| <= max|V_C|, so
    |y - y64| <= 2e-5 * max|V_C|           (fp32 output)
and a bf16 output is within one bf16 ulp of RNE(y64) plus that bound."""
import numpy as np
import pytest
import torch

from paper_2606_08094_b200 import synth

pytestmark = pytest.mark.gpu
TOL = 2e-5


@pytest.fixture(scope="module")
def vla():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    from paper_2606_08094_b200 import binding
    return binding


@pytest.fixture(scope="module")
def att():
    from oracle import attention
    return attention


def dev_bf16(bits_u16):
    return torch.from_numpy(np.ascontiguousarray(bits_u16).view(np.int16)).cuda().view(torch.bfloat16)


def run(vla, q, kc, vc, vis, Hq, Hkv, d, out_dtype):
    Mq, Mc = q.shape[0], kc.shape[0]
    out = vla.empty_out(Mq, Hq * d, out_dtype)
    out.fill_(-7.0)
    nb = vla.vla_cached_attention_workspace_bytes(Mq, Mc, Hq, Hkv, d)
    ws = torch.empty(max(nb, 16), dtype=torch.uint8, device="cuda")
    visd = None if vis is None else torch.from_numpy(vis).cuda()
    vla.vla_cached_attention(dev_bf16(q), dev_bf16(kc), dev_bf16(vc), visd, Mq, Mc, Hq, Hkv, d, out, out_dtype, ws, nb)
    torch.cuda.synchronize()
    return out


def vmax(att, vc):
    return float(np.abs(att.bf16_bits_to_f64(vc)).max())


@pytest.mark.parametrize("Mq,Mc,masked", [(16, 544, 0.0), (16, 544, 0.3), (8, 544, 0.0), (1, 544, 0.5), (50, 544, 0.2),
                                          (16, 1, 0.0), (3, 63, 0.0), (16, 64, 0.4), (5, 65, 0.0), (17, 1000, 0.9)])
def test_attention_vs_oracle_configs3_heads(vla, att, Mq, Mc, masked):
    Hq, Hkv, d = synth.ATTN_HEADS
    q, kc, vc, vis = synth.attention_inputs(Mq, Mc, Hq, Hkv, d, 7000 + Mq + Mc, masked_frac=masked)
    ref = att.cached_attention(q, kc, vc, Hq, Hkv, d, vis)
    got = run(vla, q, kc, vc, vis, Hq, Hkv, d, vla.VLA_F32).cpu().numpy().astype(np.float64)
    err = np.abs(got - ref).max()
    assert err <= TOL * vmax(att, vc), "max abs err %.3g" % err
    gb = run(vla, q, kc, vc, vis, Hq, Hkv, d, vla.VLA_BF16).float().cpu().numpy().astype(np.float64)
    ulp = np.maximum(np.abs(ref), 2.0 ** -126) * 2.0 ** -7          # >= one bf16 ulp of the reference
    assert (np.abs(gb - ref) <= ulp + TOL * vmax(att, vc)).all()


def test_all_masked_rows_and_other_head_groupings(vla, att):
    for (Hq, Hkv) in ((8, 1), (4, 4), (6, 2)):
        d, Mq, Mc = 128, 9, 130
        q, kc, vc, vis = synth.attention_inputs(Mq, Mc, Hq, Hkv, d, 7100 + Hq, masked_frac=0.5)
        vis[2] = 0
        vis[8] = 0
        ref = att.cached_attention(q, kc, vc, Hq, Hkv, d, vis)
        got = run(vla, q, kc, vc, vis, Hq, Hkv, d, vla.VLA_F32).cpu().numpy()
        assert (got[2] == 0).all() and (got[8] == 0).all() and np.isfinite(got).all()
        assert np.abs(got - ref).max() <= TOL * vmax(att, vc)


def test_large_scores_single_dominant_key(vla, att):
    Hq, Hkv, d = 4, 1, 128
    q, kc, vc, _ = synth.attention_inputs(16, 200, Hq, Hkv, d, 7200, scale=6.0)        # |scores| up to a few hundred
    ref = att.cached_attention(q, kc, vc, Hq, Hkv, d)
    got = run(vla, q, kc, vc, None, Hq, Hkv, d, vla.VLA_F32).cpu().numpy()
    assert np.isfinite(got).all()
    # the score itself is rounded in fp32 here (|s| ~ 300 -> 2^-24 * 300 * log2(e) on the exponent): 1e-4 relative
    assert np.abs(got - ref).max() <= 2e-4 * vmax(att, vc)


def test_cached_kv_from_the_ternary_linears_reused_over_solver_steps(vla, oracle, att):
    """The workload of PAPER.md lines 48-54 on configs[3] shapes: K_C, V_C = the k / v ternary linears (Eq. 4) of a 544-token
    conditioning sequence, computed ONCE, then T = 4 solver steps each with new action queries from the q linear."""
    Hq, Hkv, d = synth.ATTN_HEADS
    Mc, Mq, T = synth.ATTN_MC, 16, 4
    W = {dd["name"]: dd for dd in synth.stack_layer(0)}
    z = synth.activations(Mc, 2560, 7300)
    kc_ref = oracle.ternary_linear(z, W["k"]["w"], W["k"]["beta"], want_y64=False)["ybf16"]
    vc_ref = oracle.ternary_linear(z, W["v"]["w"], W["v"]["beta"], want_y64=False)["ybf16"]

    def lin(name, x_bits, M):
        w = W[name]
        N, K = w["w"].shape
        out = vla.empty_out(M, N, vla.VLA_BF16)
        nb = vla.vla_ternary_workspace_bytes(M, N, K)
        ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
        vla.vla_ternary_linear(vla.pack_weights(torch.from_numpy(w["w"]).cuda()), torch.tensor([float(w["beta"])], device="cuda"),
                               dev_bf16(x_bits), M, N, K, out, vla.VLA_BF16, vla.VLA_PATH_AUTO, None, None, ws, nb)
        return out
    kc_d, vc_d = lin("k", z, Mc), lin("v", z, Mc)                 # cached once
    torch.cuda.synchronize()
    assert np.array_equal(kc_d.view(torch.int16).cpu().numpy().view(np.uint16), kc_ref)
    assert np.array_equal(vc_d.view(torch.int16).cpu().numpy().view(np.uint16), vc_ref)
    nb = vla.vla_cached_attention_workspace_bytes(Mq, Mc, Hq, Hkv, d)
    ws = torch.empty(max(nb, 16), dtype=torch.uint8, device="cuda")
    for step in range(T):
        a = synth.activations(Mq, 2560, 7310 + step)
        q_ref = oracle.ternary_linear(a, W["q"]["w"], W["q"]["beta"], want_y64=False)["ybf16"]
        q_d = lin("q", a, Mq)
        out = vla.empty_out(Mq, Hq * d, vla.VLA_F32)
        vla.vla_cached_attention(q_d, kc_d, vc_d, None, Mq, Mc, Hq, Hkv, d, out, vla.VLA_F32, ws, nb)
        torch.cuda.synchronize()
        ref = att.cached_attention(q_ref, kc_ref, vc_ref, Hq, Hkv, d)
        assert np.abs(out.cpu().numpy() - ref).max() <= TOL * vmax(att, vc_ref), "step %d" % step


def test_attention_argument_errors(vla):
    q = torch.zeros((4, 20 * 128), dtype=torch.bfloat16, device="cuda")
    kv = torch.zeros((8, 5 * 128), dtype=torch.bfloat16, device="cuda")
    out = torch.zeros((4, 20 * 128), dtype=torch.float32, device="cuda")
    for bad, code in ((dict(d_k=64), vla.VLA_ERR_SHAPE), (dict(Hq=21), vla.VLA_ERR_SHAPE), (dict(Mq=0), vla.VLA_ERR_SHAPE),
                      (dict(dtype=2), vla.VLA_ERR_DTYPE)):
        a = dict(Mq=4, Mc=8, Hq=20, Hkv=5, d_k=128, dtype=0)
        a.update(bad)
        with pytest.raises(vla.VlaError) as e:
            vla.vla_cached_attention(q, kv, kv, None, a["Mq"], a["Mc"], a["Hq"], a["Hkv"], a["d_k"], out, a["dtype"], None, 0)
        assert e.value.status == code
    assert vla.vla_cached_attention_workspace_bytes(4, 8, 20, 5, 64) == 0
