"""Pins for oracle/ (CPU only).  Each test checks the oracle against something other than itself:
exact-rational brute force (tests/exact.py), the worked vector in tests/golden/, closed-form
invariants of Eq. 4, numpy/BLAS integer matmul, torch's bf16 cast.
A dropped term, wrong sign/index, transposed operand, reciprocal-multiply or round-half-away in
the oracle fails at least one of them.
"""
import itertools
import os
from fractions import Fraction

import numpy as np
import pytest
import torch

import exact
from paper_2606_08094_b200 import synth

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "worked_vector.txt")


def bf16_bits(x_f32):
    return synth._f32_to_bf16_bits(np.asarray(x_f32, np.float32))


def f32_bits(a):
    return np.asarray(a, np.float32).view(np.uint32)


def _exact_f32(bits):
    return exact.bf16_bits_to_fraction(bits >> 16) if bits & 0xFFFF == 0 else None


def f32_fraction(v):
    b = int(np.float32(v).view(np.uint32))
    e = (b >> 23) & 0xFF
    m = b & 0x7FFFFF
    s = -1 if b >> 31 else 1
    if e == 0:
        return s * Fraction(m, 1 << 23) * Fraction(2) ** (-126)
    return s * (1 + Fraction(m, 1 << 23)) * Fraction(2) ** (e - 127)


# ---------------------------------------------------------------- worked vector (tests/golden)
def _read_golden():
    d = {}
    with open(GOLDEN) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, *v = line.split()
            d[k] = [int(t, 0) for t in v]
    return d


def test_worked_vector_golden(oracle):
    g = _read_golden()
    x = np.array([g["x_bf16_bits"]], np.uint16)
    w = np.array([g["w_row0"], g["w_row1"]], np.int8)
    beta = np.array(g["beta_f32_bits"], np.uint32).view(np.float32)[0]
    r = oracle.ternary_linear(x, w, beta)
    assert r["a"].tolist() == [g["a"]]
    assert f32_bits(r["alpha"]).tolist() == g["alpha_f32_bits"]
    assert r["acc"].tolist() == [g["acc"]]
    assert f32_bits(r["y32"]).tolist() == [g["y_f32_bits"]]
    assert r["ybf16"].tolist() == [g["y_bf16_bits"]]
    # the values SURVEY.md 8(c) pin 2 prints, restated: a tie (63.5) must go to the even 64
    assert g["a"] == [64, -32, 16, 127] and g["acc"] == [175, 95]
    # within the analytic quantisation bound of the real-valued product (pin 9)
    assert abs(float(r["y32"][0, 0]) - 0.1375) < 0.05 * (2 / 127) / 2 * 3
    assert abs(float(r["y32"][0, 1]) - 0.075) < 0.05 * (2 / 127) / 2 * 3


def test_exact_constant_1e_5():
    assert float(exact.F32_1E_5) == float(np.float32(1e-5))
    assert int(np.float32(1e-5).view(np.uint32)) == 0x3727C5AC


# ---------------------------------------------------------------- brute force vs exact rationals
def test_exhaustive_weight_patterns_k4_n1(oracle):
    """All 3^4 = 81 ternary rows against python-int dot products (SURVEY 8(c) pin 1)."""
    x = bf16_bits([[0.3, -1.7, 2.2, 0.05], [5.0, 4.0, -3.0, 2.5]])
    a_ref = [exact.quant_row(r)[0] for r in x.tolist()]
    pats = list(itertools.product([-1, 0, 1], repeat=4))
    w = np.array(pats, np.int8)                     # N=81 rows at once
    r = oracle.ternary_linear(x, w, np.float32(0.05))
    assert r["a"].tolist() == a_ref
    for m in range(2):
        for n, p in enumerate(pats):
            assert int(r["acc"][m, n]) == sum(ai * wi for ai, wi in zip(a_ref[m], p))


@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_tiny_random_vs_exact(oracle, seed):
    rng = np.random.default_rng(seed)
    M, K, N = 4, 16, 4
    scale = [1.0, 1e-3, 300.0, 1e-7][seed]
    x = bf16_bits(rng.standard_normal((M, K)) * scale)
    w = rng.integers(-1, 2, (N, K)).astype(np.int8)
    beta = np.float32([0.05, 0.0123, 0.0999, 1.0][seed])
    r = oracle.ternary_linear(x, w, beta)
    e = exact.linear(x.tolist(), w.tolist(), f32_fraction(beta))
    assert r["a"].tolist() == e["a"]
    assert f32_bits(r["alpha"]).tolist() == [exact.fraction_to_f32_bits(v) for v in e["alpha"]]
    assert r["acc"].tolist() == e["acc"]
    assert f32_bits(r["y32"]).tolist() == [[exact.fraction_to_f32_bits(v) for v in row] for row in e["y32"]]
    assert r["ybf16"].tolist() == [[exact.fraction_to_bf16_bits(v) for v in row] for row in e["ybf16"]]
    # y64 is the unrounded product up to double rounding
    for m in range(M):
        for n in range(N):
            want = float(Fraction(e["acc"][m][n]) * e["alpha"][m] * f32_fraction(beta))
            assert r["y64"][m, n] == pytest.approx(want, rel=1e-14, abs=0)


def test_division_not_reciprocal_multiply(oracle):
    """Reading R1: row [0.8125, 0.40625] -> [127, 63] under true division;
    the multiply-by-(127/amax) reading gives [127, 64]."""
    x = bf16_bits([[0.8125, 0.40625]])
    a, alpha = oracle.act_quant(x)
    assert a.tolist() == [[127, 63]]
    assert exact.quant_row(x[0].tolist())[0] == [127, 63]
    recip = np.float32(127.0) / np.float32(0.8125)
    assert int(np.rint(np.float32(0.40625) * recip)) == 64      # the rejected reading differs


def test_round_half_even_not_half_away(oracle):
    # amax = 127 -> alpha = 1 exactly, so x/alpha = x and the .5 cases are exact ties
    x = bf16_bits([[127.0, 0.5, 1.5, 2.5, -0.5, -1.5, -2.5, 3.5]])
    a, alpha = oracle.act_quant(x)
    assert alpha[0] == np.float32(1.0)
    assert a.tolist() == [[127, 0, 2, 2, 0, -2, -2, 4]]


# ---------------------------------------------------------------- quantiser invariants (pin 7)
def _rows(seed, M=16, K=512, **kw):
    return synth.activations(M, K, seed, **kw)


def test_quantiser_absmax_hits_127(oracle):
    for kw in ({}, {"dist": "student_t3"}, {"outlier_frac": 0.01}):
        a, alpha = oracle.act_quant(_rows(11, **kw))
        assert (np.abs(a.astype(np.int32)).max(axis=1) == 127).all()
        assert a.min() >= -127


def test_quantiser_odd_symmetry(oracle):
    x = _rows(12)
    a, al = oracle.act_quant(x)
    a2, al2 = oracle.act_quant(x ^ np.uint16(0x8000))
    assert (a2 == -a).all() and (f32_bits(al) == f32_bits(al2)).all()


def test_quantiser_power_of_two_scale_invariance(oracle):
    x = _rows(13)
    a, al = oracle.act_quant(x)
    for k in (-5, 3, 10):
        xs = bf16_bits(oracle.bf16_to_f32(x) * np.float32(2.0 ** k))
        a2, al2 = oracle.act_quant(xs)
        assert (a2 == a).all()
        assert (al2 == al * np.float32(2.0 ** k)).all()


def test_quantiser_monotone(oracle):
    x = _rows(14, M=4, K=1024)
    a, _ = oracle.act_quant(x)
    xf = oracle.bf16_to_f32(x)
    for m in range(4):
        order = np.argsort(xf[m], kind="stable")
        assert (np.diff(a[m][order].astype(np.int32)) >= 0).all()


def test_quantiser_zero_and_tiny_rows(oracle):
    """Reading R4: an all-zero row gives a=0 and alpha = 1e-5f/127; rows below 1e-5 quantise against the floor."""
    x = np.zeros((2, 128), np.uint16)
    x[1] = bf16_bits(np.full(128, 2e-6, np.float32))
    a, alpha = oracle.act_quant(x)
    floor = np.float32(1e-5) / np.float32(127.0)
    assert (alpha == floor).all() and int(f32_bits(floor)) == exact.fraction_to_f32_bits(
        exact.round_binary(exact.F32_1E_5 / 127))
    assert (a[0] == 0).all()
    assert a[1].tolist() == exact.quant_row(x[1].tolist())[0]
    assert 0 < a[1][0] < 127


def test_quantiser_rows_vs_exact(oracle):
    x = synth.activations(3, 128, 21, outlier_frac=0.02)
    a, alpha = oracle.act_quant(x)
    for m in range(3):
        ea, eal = exact.quant_row(x[m].tolist())
        assert a[m].tolist() == ea
        assert int(f32_bits(alpha[m])) == exact.fraction_to_f32_bits(eal)


# ---------------------------------------------------------------- contraction invariants (pins 3, 4, 6, 8)
def test_unit_vector_activations_return_w_columns(oracle):
    K, N = 256, 128
    w = synth.ternary_weights(N, K, 0.35, 5)
    for c in (1.0, 0.37, 1000.0):
        x = np.zeros((K, K), np.float32)
        np.fill_diagonal(x, c)
        r = oracle.ternary_linear(bf16_bits(x), w, np.float32(1.0))
        assert (r["a"] == 127 * np.eye(K, dtype=np.int32)).all()
        assert (r["acc"] == 127 * w.T.astype(np.int32)).all()       # row j of acc = column j of W


def test_all_ones_all_zero_and_negated_w(oracle):
    x = _rows(31, M=8, K=256)
    a, _ = oracle.act_quant(x)
    N = 64
    ones = np.ones((N, 256), np.int8)
    acc = oracle.contract(a, ones)
    assert (acc == a.astype(np.int64).sum(axis=1, keepdims=True)).all()
    assert (oracle.contract(a, np.zeros((N, 256), np.int8)) == 0).all()
    w = synth.ternary_weights(N, 256, 0.33, 9)
    assert (oracle.contract(a, (-w).astype(np.int8)) == -oracle.contract(a, w)).all()


def test_linearity_and_split_k(oracle):
    x = _rows(32, M=8, K=512)
    a, _ = oracle.act_quant(x)
    w = synth.ternary_weights(96, 512, 0.35, 10)
    acc = oracle.contract(a, w)
    wp, wm = (w > 0).astype(np.int8), (w < 0).astype(np.int8)
    assert (acc == oracle.contract(a, wp) - oracle.contract(a, wm)).all()
    k1 = 192
    assert (acc == oracle.contract(a[:, :k1], w[:, :k1]) + oracle.contract(a[:, k1:], w[:, k1:])).all()


@pytest.mark.parametrize("shape_idx,M", [(0, 16), (1, 16), (2, 8), (3, 16)])
def test_contract_equals_blas_matmul_full_size(oracle, shape_idx, M):
    """O5 is an ordinary integer matrix product: float64 BLAS is exact here (|acc| <= 127*K < 2^53)."""
    p = synth.config1_point(shape_idx, M)
    a, _ = oracle.act_quant(p["x"])
    acc = oracle.contract(a, p["w"])
    ref = a.astype(np.float64) @ p["w"].T.astype(np.float64)
    assert (acc.astype(np.float64) == ref).all()
    t = torch.from_numpy(a[:2].astype(np.int32)) @ torch.from_numpy(p["w"].astype(np.int32)).T
    assert (torch.from_numpy(acc[:2]) == t).all()


def test_contract_not_transposed(oracle):
    a = np.array([[1, 2, 3, 4]], np.int8)
    w = np.array([[1, 0, 0, 0], [0, 0, 0, -1], [1, 1, 1, 1]], np.int8)      # [N=3, K=4]
    assert oracle.contract(a, w).tolist() == [[1, -4, 10]]


# ---------------------------------------------------------------- rescale, bf16, error bound
def test_rescale_order_and_groups(oracle):
    rng = np.random.default_rng(3)
    acc = rng.integers(-200000, 200000, (5, 8)).astype(np.int32)
    alpha = rng.uniform(1e-3, 0.2, 5).astype(np.float32)
    beta = np.float32(0.0371)
    y32, y64 = oracle.rescale(acc, alpha, beta)
    want = acc.astype(np.float32) * (alpha * beta)[:, None]         # numpy fp32 ops are IEEE, same order (R6)
    assert (f32_bits(y32) == f32_bits(want)).all()
    assert np.allclose(y64, acc.astype(np.float64) * alpha.astype(np.float64)[:, None] * float(beta), rtol=1e-15)
    assert (np.abs(y32 - y64) <= 1e-6 * np.abs(y64)).all()
    bg = np.array([0.01, 0.09], np.float32)                          # two output groups of 4 channels
    yg, _ = oracle.rescale(acc, alpha, bg)
    assert (f32_bits(yg[:, :4]) == f32_bits(acc[:, :4].astype(np.float32) * (alpha * bg[0])[:, None])).all()
    assert (f32_bits(yg[:, 4:]) == f32_bits(acc[:, 4:].astype(np.float32) * (alpha * bg[1])[:, None])).all()


def test_ternary_linear_bf16_with_three_output_groups_vs_exact(oracle):
    """orc_ternary_linear's bf16 output with a [G=3] beta vector (oracle.cpp, the grouped branch): every group's
    channels against tests/exact.py (exact rationals, own rounding), which knows nothing about groups -- it is called
    once per group with that group's scalar beta."""
    rng = np.random.default_rng(77)
    M, K, N, G = 3, 16, 6, 3
    x_bits = synth.activations(M, K, 991, outlier_frac=0.1)
    w = rng.integers(-1, 2, (N, K)).astype(np.int8)
    betas = np.array([0.0371, 0.5, 0.011], np.float32)
    got = oracle.ternary_linear(x_bits, w, betas)
    per = N // G
    for g in range(G):
        ex = exact.linear([list(map(int, r)) for r in x_bits], [list(map(int, r)) for r in w[g * per:(g + 1) * per]],
                          Fraction(float(betas[g])))
        for m in range(M):
            for n in range(per):
                assert int(got["acc"][m, g * per + n]) == ex["acc"][m][n]
                assert int(f32_bits(got["y32"])[m, g * per + n]) == exact.fraction_to_f32_bits(ex["y32"][m][n])
                assert int(got["ybf16"][m, g * per + n]) == exact.fraction_to_bf16_bits(ex["ybf16"][m][n])
    # and it is NOT what a single scale would give
    one = oracle.ternary_linear(x_bits, w, betas[:1])
    assert not np.array_equal(one["ybf16"][:, per:], got["ybf16"][:, per:])


def test_bf16_rne_matches_torch_and_ties(oracle):
    rng = np.random.default_rng(4)
    v = (rng.standard_normal(200000) * np.exp(rng.uniform(-20, 20, 200000))).astype(np.float32)
    ties = np.array([0x3F808000, 0x3F818000, 0xBF808000, 0x3F80FFFF, 0x3F808001, 0x00000000, 0x80000000],
                    np.uint32).view(np.float32)
    v = np.concatenate([v, ties])
    got = oracle.f32_to_bf16(v)
    want = torch.from_numpy(v).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert (got == want).all()
    assert got[-7:-2].tolist() == [0x3F80, 0x3F82, 0xBF80, 0x3F81, 0x3F81]   # even, even, even, up, up
    assert (oracle.bf16_to_f32(got).view(np.uint32) == (got.astype(np.uint32) << 16)).all()


def test_error_bound_vs_float_gemm(oracle):
    """|y - beta*sum_j x_j w_nj| <= beta*(alpha_m/2)*nnz(w_n)   (SURVEY 8(c) pin 9)."""
    p = synth.config0()
    r = oracle.ternary_linear(p["x"], p["w"], p["beta"])
    xf = oracle.bf16_to_f32(p["x"]).astype(np.float64)
    real = float(p["beta"]) * xf @ p["w"].T.astype(np.float64)
    nnz = (p["w"] != 0).sum(axis=1)
    bound = float(p["beta"]) * (r["alpha"].astype(np.float64)[:, None] / 2) * nnz[None, :]
    assert (np.abs(r["y64"] - real) <= bound * (1 + 1e-6) + 1e-12).all()
    assert np.abs(r["y64"] - real).max() > 0


def test_pack_ref_round_trip(oracle):
    w = synth.ternary_weights(64, 128, 0.35, 77)
    packed, bad = oracle.pack_ref(w)
    assert bad == 0 and packed.size == w.size // 4
    assert (oracle.unpack_ref(packed, w.shape) == w).all()
    w2 = w.copy()
    w2[3, 5] = 2
    assert oracle.pack_ref(w2)[1] == 1


def test_full_path_composition(oracle):
    p = synth.config1_point(1, 8)
    r = oracle.ternary_linear(p["x"], p["w"], p["beta"])
    a, alpha = oracle.act_quant(p["x"])
    acc = oracle.contract(a, p["w"])
    y32, y64 = oracle.rescale(acc, alpha, p["beta"])
    assert (r["a"] == a).all() and (r["acc"] == acc).all()
    assert (f32_bits(r["y32"]) == f32_bits(y32)).all()
    assert (r["ybf16"] == oracle.f32_to_bf16(y32)).all()
