"""Oracle of the cached-conditioning cross-attention, Eq. 2 of arxiv/paper_2606_08094 (section
III-B) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may
import this module; it shares no code with the CUDA path.

    Attn(Q, K_C, V_C; M) = softmax(Q K_C^T / sqrt(d_k) + M) V_C                      (Eq. 2, one head)

"Q contains action queries ... d_k is the key dimension.  The additive mask M is zero for visible keys and -inf for
masked keys.  Softmax operates over keys.".  K_C = Z W_K and V_C = Z W_V are CACHED projections of the
conditioning sequence: here they are inputs (the k / v ternary linears of Eq. 4 produce them).

The definition is written out in float64 on the exact values of the bf16 inputs, one head at a time, with plain numpy:
no blocking, no online softmax, no fusion.  Readings where the paper is silent (R14-R16):
  R14  grouped-query heads: query head h reads key/value head h // (n_q_heads // n_kv_heads)   (BASELINE.json configs[3]:
       20 query / 5 KV heads; the paper's Eq. 2 "describes one attention head")
  R15  a query row whose keys are ALL masked has no softmax (0/0): its output is defined as 0
  R16  the mask is carried as visibility bytes (1 = visible: M = 0; 0 = masked: M = -inf); NULL = everything visible
"""
import numpy as np


def bf16_bits_to_f64(bits_u16):
    """exact value of bf16 bit patterns (uint16) as float64"""
    b = np.ascontiguousarray(bits_u16, dtype=np.uint16)
    return (b.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def cached_attention(q_bits, kc_bits, vc_bits, n_q_heads, n_kv_heads, d_k, visible=None):
    """q_bits [Mq, n_q_heads*d_k], kc_bits / vc_bits [Mc, n_kv_heads*d_k]: bf16 bit patterns (uint16);
    visible: None or uint8 [Mq, Mc] (1 = visible).  Returns float64 [Mq, n_q_heads*d_k]."""
    q = bf16_bits_to_f64(q_bits)
    kc = bf16_bits_to_f64(kc_bits)
    vc = bf16_bits_to_f64(vc_bits)
    Mq, Mc = q.shape[0], kc.shape[0]
    assert q.shape[1] == n_q_heads * d_k and kc.shape[1] == n_kv_heads * d_k and vc.shape == kc.shape
    assert n_q_heads % n_kv_heads == 0
    group = n_q_heads // n_kv_heads
    out = np.zeros((Mq, n_q_heads * d_k), np.float64)
    for h in range(n_q_heads):
        g = h // group                                            # R14
        Q = q[:, h * d_k:(h + 1) * d_k]
        K = kc[:, g * d_k:(g + 1) * d_k]
        V = vc[:, g * d_k:(g + 1) * d_k]
        S = (Q @ K.T) / np.sqrt(np.float64(d_k))                  # Q K_C^T / sqrt(d_k)
        for m in range(Mq):
            s = S[m].copy()
            if visible is not None:
                s[visible[m] == 0] = -np.inf                      # + M
            if not np.isfinite(s).any():
                continue                                          # R15: all keys masked -> 0
            e = np.exp(s - s.max())                               # softmax over keys (shift-invariant form)
            p = e / e.sum()
            out[m, h * d_k:(h + 1) * d_k] = p @ V
    return out
