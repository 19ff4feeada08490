"""Pins of the attention oracle (oracle/attention.py, Eq. 2 of the paper) against what the
mathematics fixes: brute force in pure Python, closed forms (one key, two keys, zero queries, equal keys), invariants
(masked keys are irrelevant, key permutation, no overflow), the grouped-query head map (R14), the all-masked
rule (R15) and scipy's softmax at the configs[3] shape.  No GPU."""
import math

import numpy as np
import pytest

from oracle import attention as att
from paper_2606_08094_b200 import synth


def f64(bits):
    return att.bf16_bits_to_f64(bits)


def brute(q, kc, vc, Hq, Hkv, d, vis):
    """Eq. 2 with Python floats and loops only"""
    Mq, Mc = q.shape[0], kc.shape[0]
    out = [[0.0] * (Hq * d) for _ in range(Mq)]
    for h in range(Hq):
        g = h // (Hq // Hkv)
        for m in range(Mq):
            s = []
            for j in range(Mc):
                if vis is not None and vis[m][j] == 0:
                    s.append(None)
                    continue
                dot = 0.0
                for i in range(d):
                    dot += float(q[m][h * d + i]) * float(kc[j][g * d + i])
                s.append(dot / math.sqrt(d))
            live = [v for v in s if v is not None]
            if not live:
                continue
            mx = max(live)
            w = [0.0 if v is None else math.exp(v - mx) for v in s]
            z = sum(w)
            for i in range(d):
                out[m][h * d + i] = sum(w[j] * float(vc[j][g * d + i]) for j in range(Mc)) / z
    return np.array(out)


@pytest.mark.parametrize("seed,masked", [(1, 0.0), (2, 0.4), (3, 0.7)])
def test_brute_force_tiny(seed, masked):
    Hq, Hkv, d = 4, 2, 8
    q, kc, vc, vis = synth.attention_inputs(3, 7, Hq, Hkv, d, seed, masked_frac=masked)
    got = att.cached_attention(q, kc, vc, Hq, Hkv, d, vis)
    want = brute(f64(q), f64(kc), f64(vc), Hq, Hkv, d, vis)
    assert np.allclose(got, want, rtol=1e-12, atol=1e-14)


def test_single_visible_key_returns_its_value_row():
    Hq, Hkv, d = 2, 1, 16
    q, kc, vc, _ = synth.attention_inputs(4, 9, Hq, Hkv, d, 5)
    vis = np.zeros((4, 9), np.uint8)
    vis[np.arange(4), [0, 3, 8, 5]] = 1
    got = att.cached_attention(q, kc, vc, Hq, Hkv, d, vis)
    v = f64(vc)
    for m, j in enumerate([0, 3, 8, 5]):
        for h in range(Hq):
            assert np.array_equal(got[m, h * d:(h + 1) * d], v[j])


def test_two_keys_closed_form_sigmoid():
    """two keys: out = sigma(D) v1 + (1 - sigma(D)) v2, D = q.(k1 - k2) / sqrt(d): catches a dropped scale, a wrong
    sign and softmax over the wrong axis"""
    Hq, Hkv, d = 1, 1, 32
    q, kc, vc, _ = synth.attention_inputs(5, 2, Hq, Hkv, d, 6)
    got = att.cached_attention(q, kc, vc, Hq, Hkv, d)
    Q, K, V = f64(q), f64(kc), f64(vc)
    for m in range(5):
        D = float(Q[m] @ (K[0] - K[1])) / math.sqrt(d)
        sg = 1.0 / (1.0 + math.exp(-D))
        assert np.allclose(got[m], sg * V[0] + (1.0 - sg) * V[1], rtol=1e-13, atol=1e-15)


def test_zero_queries_and_equal_keys_give_the_mean_of_visible_values():
    Hq, Hkv, d = 2, 2, 8
    q, kc, vc, vis = synth.attention_inputs(3, 11, Hq, Hkv, d, 7, masked_frac=0.3)
    V = f64(vc)
    got = att.cached_attention(np.zeros_like(q), kc, vc, Hq, Hkv, d, vis)
    for m in range(3):
        for h in range(Hq):
            want = V[vis[m] == 1][:, h * d:(h + 1) * d].mean(axis=0)
            assert np.allclose(got[m, h * d:(h + 1) * d], want, rtol=1e-13)
    kc_same = np.repeat(kc[:1], 11, axis=0)
    got2 = att.cached_attention(q, kc_same, vc, Hq, Hkv, d, vis)
    assert np.allclose(got2, got, rtol=1e-13)


def test_masked_keys_are_irrelevant_and_keys_permute():
    Hq, Hkv, d = 4, 1, 16
    q, kc, vc, vis = synth.attention_inputs(6, 13, Hq, Hkv, d, 8, masked_frac=0.5)
    base = att.cached_attention(q, kc, vc, Hq, Hkv, d, vis)
    kc2, vc2 = kc.copy(), vc.copy()
    dead = np.where(vis.sum(axis=0) == 0)[0]
    kc2[dead] = 0x7F00                                            # huge finite bf16 in rows nobody sees
    vc2[dead] = 0xFF00
    assert np.array_equal(att.cached_attention(q, kc2, vc2, Hq, Hkv, d, vis), base)
    for m in range(6):                                            # equals attention over the visible subset alone
        keep = vis[m] == 1
        sub = att.cached_attention(q[m:m + 1], kc[keep], vc[keep], Hq, Hkv, d)
        assert np.allclose(sub[0], base[m], rtol=1e-13)
    perm = np.random.default_rng(0).permutation(13)
    assert np.allclose(att.cached_attention(q, kc[perm], vc[perm], Hq, Hkv, d, vis[:, perm]), base, rtol=1e-12)


def test_grouped_query_head_map_and_all_masked_rows():
    Hq, Hkv, d = 6, 3, 8                                          # R14: query heads 0,1 -> kv 0; 2,3 -> kv 1; 4,5 -> kv 2
    q, kc, vc, _ = synth.attention_inputs(2, 5, Hq, Hkv, d, 9)
    got = att.cached_attention(q, kc, vc, Hq, Hkv, d)
    for h in range(Hq):
        g = h // 2
        one = att.cached_attention(q[:, h * d:(h + 1) * d], kc[:, g * d:(g + 1) * d], vc[:, g * d:(g + 1) * d], 1, 1, d)
        assert np.array_equal(one, got[:, h * d:(h + 1) * d])
    vis = np.ones((2, 5), np.uint8)
    vis[1] = 0                                                    # R15: nothing visible -> zeros, no NaN
    z = att.cached_attention(q, kc, vc, Hq, Hkv, d, vis)
    assert np.array_equal(z[1], np.zeros(Hq * d)) and np.isfinite(z).all() and np.array_equal(z[0], got[0])


def test_dominant_key_and_huge_scores_do_not_overflow():
    Hq, Hkv, d = 1, 1, 128
    q, kc, vc, _ = synth.attention_inputs(2, 6, Hq, Hkv, d, 10, scale=60.0)      # scores of order 1e4
    got = att.cached_attention(q, kc, vc, Hq, Hkv, d)
    assert np.isfinite(got).all()
    S = f64(q) @ f64(kc).T / math.sqrt(d)
    for m in range(2):
        j = int(S[m].argmax())
        if S[m, j] - np.partition(S[m], -2)[-2] > 50:             # the runner-up weighs < e^-50
            assert np.allclose(got[m], f64(vc)[j], rtol=1e-12)


def test_scipy_softmax_at_the_configs3_shape():
    from scipy.special import softmax
    Hq, Hkv, d = synth.ATTN_HEADS
    q, kc, vc, vis = synth.attention_inputs(16, synth.ATTN_MC, Hq, Hkv, d, 11, masked_frac=0.1)
    got = att.cached_attention(q, kc, vc, Hq, Hkv, d, vis)
    Q, K, V = f64(q), f64(kc), f64(vc)
    for h in (0, 7, 19):
        g = h // (Hq // Hkv)
        S = Q[:, h * d:(h + 1) * d] @ K[:, g * d:(g + 1) * d].T / math.sqrt(d)
        S[vis == 0] = -np.inf
        want = softmax(S, axis=1) @ V[:, g * d:(g + 1) * d]
        assert np.allclose(got[:, h * d:(h + 1) * d], want, rtol=1e-12, atol=1e-14)
