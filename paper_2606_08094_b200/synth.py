"""Seeded synthetic inputs for BASELINE.json's configs (recipe: DESIGN.md "Input recipe").

This module serves both the CUDA path and the oracle and therefore holds NONE of the method's
arithmetic (no quantiser, no packing, no contraction): it only draws ternary weights, bf16
activations and scales with the shapes and distributions BASELINE.json:configs names.  The
BitVLA checkpoint and LIBERO episodes the paper measured on are not available; these
arrays stand in for them.

bf16 is carried as uint16 bit patterns (numpy has no bf16); the fp32 -> bf16 cast of the drawn
samples uses torch's CPU cast.
"""
import math

import numpy as np
import torch

# (K, N) of the four BitNet-2B-class linears (BASELINE.json configs[1..3]) and the sweep's extra shape.
MODEL_SHAPES = [(2560, 2560), (2560, 640), (2560, 6912), (6912, 2560)]
SWEEP_SHAPES = [(2560, 2560), (2560, 6912), (6912, 2560), (8192, 8192)]
SWEEP_M = [1 << i for i in range(13)]
SWEEP_ZERO_FRAC = [0.2, 0.33, 0.5]
SWEEP_DISTS = ["gauss", "student_t3"]
DECODE_M = [1, 8, 16]
PREFILL_M = 544          # 2 cameras x 256 vision tokens + 32 text tokens (configs[2])
STACK_LAYERS = 30
# (name, K, N) of one decoder layer's ternary linears in execution order (configs[3]):
# hidden 2560, 20 query / 5 KV heads of dim 128, FFN 6912.
STACK_LINEARS = [("q", 2560, 2560), ("k", 2560, 640), ("v", 2560, 640), ("o", 2560, 2560),
                 ("gate", 2560, 6912), ("up", 2560, 6912), ("down", 6912, 2560)]


def _f32_to_bf16_bits(x_f32):
    t = torch.from_numpy(np.ascontiguousarray(x_f32, dtype=np.float32)).to(torch.bfloat16)
    return t.view(torch.int16).numpy().view(np.uint16).copy()


def ternary_weights(N, K, p_zero, seed):
    """int8 [N,K], i.i.d. with P(0)=p_zero and P(+1)=P(-1)=(1-p_zero)/2."""
    rng = np.random.Generator(np.random.PCG64(seed))
    u = rng.random((N, K), dtype=np.float32)
    half = (1.0 - p_zero) / 2.0
    w = np.zeros((N, K), np.int8)
    w[u < half] = -1
    w[u >= 1.0 - half] = 1
    return w


def activations(M, K, seed, dist="gauss", outlier_frac=0.0, outlier_scale=20.0):
    """bf16 bit patterns, uint16 [M,K].  dist: "gauss" N(0,1) or "student_t3" (nu=3).
    outlier_frac > 0 multiplies ceil(outlier_frac*K) channel indices (fixed across tokens) by
    outlier_scale before the bf16 cast (configs[1]: 1 % outlier channels x20)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    if dist == "gauss":
        x = rng.standard_normal((M, K), dtype=np.float32)
    elif dist == "student_t3":
        x = rng.standard_t(3.0, (M, K)).astype(np.float32)
    else:
        raise ValueError(dist)
    if outlier_frac > 0.0:
        n_out = int(math.ceil(outlier_frac * K))
        idx = rng.choice(K, size=n_out, replace=False)
        x[:, idx] *= np.float32(outlier_scale)
    return _f32_to_bf16_bits(x)


def weight_scale(seed, lo=0.01, hi=0.1):
    rng = np.random.Generator(np.random.PCG64(seed))
    return np.float32(rng.uniform(lo, hi))


def _seed_w(c, shape_idx, zf_idx=0):
    return 1000 * c + 10 * shape_idx + zf_idx


def _seed_x(c, shape_idx, dist_idx=0):
    return 500_000 + 1000 * c + 10 * shape_idx + dist_idx


def config0():
    """configs[0]: M=8, K=256, N=256, P(0)=1/3, beta=0.05, X ~ N(0,1) bf16, fp32 out, seed 0."""
    return dict(name="C0", M=8, K=256, N=256, w=ternary_weights(256, 256, 1.0 / 3.0, 0),
                beta=np.float32(0.05), x=activations(8, 256, 0), out="f32")


def config1_point(shape_idx, M):
    """configs[1]: decode / action chunk, bf16 out.  Rows are drawn at max M=16 and sliced."""
    K, N = MODEL_SHAPES[shape_idx]
    x = activations(max(DECODE_M), K, _seed_x(1, shape_idx), outlier_frac=0.01)[:M]
    return dict(name="C1", M=M, K=K, N=N, w=ternary_weights(N, K, 0.35, _seed_w(1, shape_idx)),
                beta=weight_scale(_seed_w(1, shape_idx) + 7), x=np.ascontiguousarray(x), out="bf16")


def config2_point(shape_idx, M=PREFILL_M):
    """configs[2]: prefill at M=544, quant fused into the call, fp32 out."""
    K, N = MODEL_SHAPES[shape_idx]
    return dict(name="C2", M=M, K=K, N=N, w=ternary_weights(N, K, 0.35, _seed_w(2, shape_idx)),
                beta=weight_scale(_seed_w(2, shape_idx) + 7),
                x=activations(M, K, _seed_x(2, shape_idx), outlier_frac=0.01), out="f32")


def stack_layer(layer):
    """configs[3]: the 7 ternary linears of decoder layer `layer`.  beta = 1/sqrt(0.65*K) keeps the
    chained activations at unit scale (reading R12)."""
    out = []
    for i, (name, K, N) in enumerate(STACK_LINEARS):
        out.append(dict(name=name, K=K, N=N, w=ternary_weights(N, K, 0.35, 3000 + 10 * layer + i),
                        beta=np.float32(1.0 / math.sqrt(0.65 * K))))
    return out


def stack_input(M):
    return activations(M, 2560, _seed_x(3, 0))


def config4_point(M, shape_idx, zf_idx, dist_idx):
    """configs[4]: roofline sweep point; beta=0.05, fused quant, fp32 out."""
    K, N = SWEEP_SHAPES[shape_idx]
    return dict(name="C4", M=M, K=K, N=N,
                w=ternary_weights(N, K, SWEEP_ZERO_FRAC[zf_idx], _seed_w(4, shape_idx, zf_idx)),
                beta=np.float32(0.05),
                x=np.ascontiguousarray(
                    activations(max(SWEEP_M), K, _seed_x(4, shape_idx, dist_idx),
                                dist=SWEEP_DISTS[dist_idx])[:M]),
                out="f32")


# ------------------------------------------------------------------ cached-conditioning attention
ATTN_HEADS = (20, 5, 128)      # query heads, KV heads, head dim of BASELINE.json configs[3]
ATTN_MC = PREFILL_M            # conditioning tokens: the 544-token prefix of configs[2]


def attention_inputs(Mq, Mc, n_q_heads, n_kv_heads, d_k, seed, masked_frac=0.0, scale=1.0):
    """bf16 bit patterns of Q [Mq, Hq*d], K_C / V_C [Mc, Hkv*d] (N(0, scale^2), stand-ins for the outputs of the q / k / v
    linears on LIBERO observations, which are not available) and a visibility mask uint8 [Mq, Mc] (1 = visible; with
    masked_frac > 0 a random subset of keys is masked per query row, at least one key stays visible), or None."""
    rng = np.random.Generator(np.random.PCG64(seed))
    q = _f32_to_bf16_bits(rng.standard_normal((Mq, n_q_heads * d_k), dtype=np.float32) * np.float32(scale))
    kc = _f32_to_bf16_bits(rng.standard_normal((Mc, n_kv_heads * d_k), dtype=np.float32) * np.float32(scale))
    vc = _f32_to_bf16_bits(rng.standard_normal((Mc, n_kv_heads * d_k), dtype=np.float32))
    vis = None
    if masked_frac > 0.0:
        vis = (rng.random((Mq, Mc)) >= masked_frac).astype(np.uint8)
        vis[np.arange(Mq), rng.integers(0, Mc, Mq)] = 1
    return q, kc, vc, vis
