"""GPU parity tests (-m gpu) of the persistent program kernel (vla_program_build / vla_program_run): lists of
small-M ternary linears, independent and chained, against the CPU oracle.  Same bars as test_gpu_parity.py;
because the canonical operation order is followed (R1, R6) every output is also bit-identical, which
is what makes the free-running chained stack of BASELINE.json configs[3] checkable end to end.
"""
import numpy as np
import pytest
import torch

from paper_2606_08094_b200 import synth

pytestmark = pytest.mark.gpu

REL_TOL_F32 = 1e-6


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


def bits(t):
    return t.view(torch.int16).cpu().numpy().view(np.uint16)


_TDT = {0: torch.float32, 1: torch.bfloat16, 2: torch.int32}


def make_point(vla, M, K, N, seed, dtype, p_zero=0.35, want_xq=False):
    w = synth.ternary_weights(N, K, p_zero, seed)
    x = synth.activations(M, K, seed + 1, outlier_frac=0.01)
    beta = synth.weight_scale(seed + 2)
    d = dict(M=M, K=K, N=N, w=w, x_bits=x, beta=beta, dtype=dtype, packed=vla.pack_weights(dev(w)),
             beta_d=dev(np.array([beta], np.float32)), x=dev_bf16(x),
             out=torch.full((M, N), -7, dtype=_TDT[dtype], device="cuda"))
    if want_xq:
        d["xq"] = torch.full((M, K), 99, dtype=torch.int8, device="cuda")
        d["xs"] = torch.full((M,), -1.0, dtype=torch.float32, device="cuda")
    return d


def stage_of(p):
    return dict(x=p["x"], M=p["M"], K=p["K"], depends=0, xq_opt=p.get("xq"), x_scale_opt=p.get("xs"),
                linears=[dict(packed=p["packed"], w_scale=p["beta_d"], out=p["out"], N=p["N"], out_dtype=p["dtype"])])


def check_point(vla, oracle, p):
    ref = oracle.ternary_linear(p["x_bits"], p["w"], p["beta"])
    if p["dtype"] == vla.VLA_I32:
        got = p["out"].cpu().numpy()
        bad = np.argwhere(got != ref["acc"])
        assert bad.size == 0, "int32 differs at %d places, first %s" % (len(bad), bad[0])
    elif p["dtype"] == vla.VLA_F32:
        got = p["out"].cpu().numpy()
        assert np.all(np.abs(got.astype(np.float64) - ref["y64"]) <= REL_TOL_F32 * np.abs(ref["y64"]))
        assert np.array_equal(got.view(np.uint32), ref["y32"].view(np.uint32))
    else:
        assert np.array_equal(bits(p["out"]), ref["ybf16"])
    if "xq" in p:
        assert np.array_equal(p["xq"].cpu().numpy(), ref["a"])
        assert np.array_equal(p["xs"].cpu().numpy().view(np.uint32), ref["alpha"].view(np.uint32))


@pytest.mark.parametrize("M,K,N", [(1, 128, 128), (8, 256, 256), (3, 384, 128), (16, 2560, 640), (13, 4224, 256),
                                   (8, 8192, 384), (16, 8192, 128), (5, 6912, 2560)])
@pytest.mark.parametrize("dtype", [0, 1, 2])
def test_single_stage_program(vla, oracle, M, K, N, dtype):
    """one linear per program, every output type; shapes span 1..4 ring chunks, ragged piece counts, both M tiles"""
    p = make_point(vla, M, K, N, 9000 + M + K + N, dtype, want_xq=True)
    prog = vla.compile_program([stage_of(p)])
    vla.vla_program_run(prog)
    torch.cuda.synchronize()
    check_point(vla, oracle, p)
    vla.vla_program_release(prog)


def test_configs1_as_one_program(vla, oracle):
    """BASELINE.json configs[1]: the 12 decode points (4 shapes x M in {1,8,16}) as 12 independent stages of ONE
    launch, at full size, in the launch configuration bench.py times; run twice (the counters reset themselves)
    and once from a CUDA graph."""
    pts = []
    for M in synth.DECODE_M:
        for si in range(len(synth.MODEL_SHAPES)):
            c = synth.config1_point(si, M)
            pts.append(dict(M=M, K=c["K"], N=c["N"], w=c["w"], x_bits=c["x"], beta=c["beta"], dtype=vla.VLA_BF16,
                            packed=vla.pack_weights(dev(c["w"])), beta_d=dev(np.array([c["beta"]], np.float32)),
                            x=dev_bf16(c["x"]), out=torch.zeros((M, c["N"]), dtype=torch.bfloat16, device="cuda")))
    prog = vla.compile_program([stage_of(p) for p in pts])
    for rep in range(2):
        for p in pts:
            p["out"].fill_(-3.0)
        vla.vla_program_run(prog)
        torch.cuda.synchronize()
        for p in pts:
            check_point(vla, oracle, p)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        vla.vla_program_run(prog)
        vla.vla_program_run(prog)
    for p in pts:
        p["out"].fill_(-3.0)
    g.replay()
    torch.cuda.synchronize()
    for p in pts:
        check_point(vla, oracle, p)


def oracle_stack(oracle, weights, x_bits):
    """The chain of DESIGN.md R12 on the oracle, free-running, all intermediates bf16.  Returns per layer the
    bf16 bit patterns of q, k, v, o, gate, up, down."""
    outs = []
    h = x_bits
    for lw in weights:
        W = {d["name"]: d for d in lw}
        o = {}
        for n in ("q", "k", "v"):
            o[n] = oracle.ternary_linear(h, W[n]["w"], W[n]["beta"], want_y64=False)["ybf16"]
        o["o"] = oracle.ternary_linear(o["q"], W["o"]["w"], W["o"]["beta"], want_y64=False)["ybf16"]
        for n in ("gate", "up"):
            o[n] = oracle.ternary_linear(o["o"], W[n]["w"], W[n]["beta"], want_y64=False)["ybf16"]
        o["down"] = oracle.ternary_linear(o["up"], W["down"]["w"], W["down"]["beta"], want_y64=False)["ybf16"]
        outs.append(o)
        h = o["down"]
    return outs


@pytest.mark.parametrize("M", [1, 8, 16])
def test_chained_stack_free_running(vla, oracle, M):
    """configs[3] layers (full shapes: hidden 2560, 5 KV heads x 128, FFN 6912), 3 layers = 12 dependent stages in
    one launch; every intermediate of every layer must be bit-identical to the oracle's chain."""
    from paper_2606_08094_b200.stack import Stack
    layers = 3
    weights = [synth.stack_layer(l) for l in range(layers)]
    x = synth.stack_input(M)
    st = Stack(layers, M, weights=weights)
    st.set_input(x)
    st.compile()
    for rep in range(2):
        st.run_program()
        torch.cuda.synchronize()
        ref = oracle_stack(oracle, weights, x)
        for l in range(layers):
            for n in ref[l]:
                assert np.array_equal(bits(st.out[l][n]), ref[l][n]), "layer %d %s differs (rep %d)" % (l, n, rep)
    # the per-call route (quant kernel + one GEMM launch per linear) must give the same bits
    st2 = Stack(layers, M, weights=weights)
    st2.set_input(x)
    st2.alloc_call_workspace()
    st2.run_stack_calls()
    torch.cuda.synchronize()
    for l in range(layers):
        for n in ref[l]:
            assert np.array_equal(bits(st2.out[l][n]), ref[l][n]), "per-call route: layer %d %s differs" % (l, n)


@pytest.mark.parametrize("M,K,N,nst", [(16, 8192, 2048, 16), (8, 6912, 1024, 16), (16, 6912, 2048, 16), (5, 8192, 1536, 12)])
def test_team_mode_with_multi_chunk_granules(vla, oracle, M, K, N, nst):
    """Granules longer than one ring slot (K = 6912: two chunks, K = 8192: three) in TEAM mode with as few as three ring
    slots (M = 16 leaves the ring what 16*K bytes of activations do not take): `nst` independent stages share one
    weight tensor and one activation matrix, so every group is ~9 CTAs with >= 3 granules each, and every team runs
    several granules through its own slots.  (A team that waited two mbarrier phases ahead of a slot read stale chunks.)"""
    w = synth.ternary_weights(N, K, 0.35, 4242 + K + N)
    x_bits = synth.activations(M, K, 4243, outlier_frac=0.01)
    beta = synth.weight_scale(4244)
    packed = vla.pack_weights(dev(w))
    beta_d = dev(np.array([beta], np.float32))
    x = dev_bf16(x_bits)
    outs = [torch.full((M, N), -7, dtype=torch.int32 if c % 2 else torch.bfloat16, device="cuda") for c in range(nst)]
    stages = [dict(x=x, M=M, K=K, depends=0,
                   linears=[dict(packed=packed, w_scale=beta_d, out=outs[c], N=N, out_dtype=2 if c % 2 else 1)]) for c in range(nst)]
    prog = vla.compile_program(stages)
    ref = oracle.ternary_linear(x_bits, w, beta)
    for rep in range(2):
        vla.vla_program_run(prog)
        torch.cuda.synchronize()
        for c in range(nst):
            if c % 2:
                assert np.array_equal(outs[c].cpu().numpy(), ref["acc"]), "stage %d int32 (rep %d)" % (c, rep)
            else:
                assert np.array_equal(bits(outs[c]), ref["ybf16"]), "stage %d bf16 (rep %d)" % (c, rep)
    vla.vla_program_release(prog)


def test_chained_stack_m544_grouped_tcgen05(vla, oracle):
    """configs[3] at M=544, the launch configuration `bench.py --workload stack` times: 3 full-size layers through
    Stack.run_stack_calls (activation quant + ONE grouped tcgen05 launch per stage: q|k|v as N=3840, gate|up as N=13824,
    channel tiles crossing the linears' boundaries inside one persistent tile walk), free-running, every intermediate of
    every layer bit-identical to the oracle's chain."""
    from paper_2606_08094_b200.stack import Stack
    layers, M = 3, synth.PREFILL_M
    weights = [synth.stack_layer(l) for l in range(layers)]
    x = synth.stack_input(M)
    st = Stack(layers, M, weights=weights)
    st.set_input(x)
    st.alloc_call_workspace()
    st.run_stack_calls()
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()                               # and once more from a CUDA graph, as the bench runs it
    with torch.cuda.graph(g):
        st.run_stack_calls()
    ref = oracle_stack(oracle, weights, x)
    for rep in range(2):
        for l in range(layers):
            for n in ref[l]:
                assert np.array_equal(bits(st.out[l][n]), ref[l][n]), "layer %d %s differs (rep %d)" % (l, n, rep)
                st.out[l][n].zero_()
        if rep == 0:
            g.replay()
            torch.cuda.synchronize()


def test_full_depth_stack_m8_one_launch(vla, oracle):
    """The launch `bench.py --workload stack` times at M=8: all 30 layers = 120 dependent phases, 210 linears, in ONE
    persistent launch (descriptor tables near their capacity), free-running against the oracle's 30-layer chain."""
    from paper_2606_08094_b200.stack import Stack
    layers, M = synth.STACK_LAYERS, 8
    weights = [synth.stack_layer(l) for l in range(layers)]
    x = synth.stack_input(M)
    st = Stack(layers, M, weights=weights)
    st.set_input(x)
    st.compile()
    ref = oracle_stack(oracle, weights, x)
    for rep in range(2):
        st.run_program()
        torch.cuda.synchronize()
        for l in range(layers):
            for n in ref[l]:
                assert np.array_equal(bits(st.out[l][n]), ref[l][n]), "layer %d %s differs (rep %d)" % (l, n, rep)


def test_program_errors(vla):
    p = make_point(vla, 8, 256, 256, 5, vla.VLA_BF16)
    bad_m = dict(stage_of(p), M=0)
    assert vla.vla_program_bytes([bad_m]) == 0
    mixed = [stage_of(p), dict(stage_of(p), M=17)]      # M > 16 is a LARGE program (test_gpu_lprogram.py): one kind per program
    assert vla.vla_program_bytes(mixed) == 0
    bad_k = dict(stage_of(p), K=8192 + 128)
    assert vla.vla_program_bytes([bad_k]) == 0
    with pytest.raises(vla.VlaError) as e:
        vla.vla_program_run(p["out"])          # not a compiled program
    assert e.value.status == vla.VLA_ERR_VALUE


def test_mixed_phases_and_token_counts(vla, oracle):
    """Phase 0: two independent stages (M=8 and M=3); phase 1: a stage that reads phase 0's bf16 output (depends=1)
    plus an independent M=16 stage that joins it; phase 2: another dependent stage.  Every output vs the oracle."""
    def lin(N, K, seed, dt=1):
        w = synth.ternary_weights(N, K, 0.35, seed)
        beta = synth.weight_scale(seed + 1)
        return dict(w=w, beta=beta, packed=vla.pack_weights(dev(w)), beta_d=dev(np.array([beta], np.float32)), N=N, K=K, dt=dt)
    xa = synth.activations(8, 256, 11)
    xb = synth.activations(3, 512, 12, outlier_frac=0.01)
    xd = synth.activations(16, 128, 13)
    A, B, C, D, E_ = lin(384, 256, 21), lin(128, 512, 22, dt=0), lin(256, 384, 23), lin(640, 128, 24, dt=2), lin(128, 256, 25, dt=0)
    ya = torch.zeros((8, 384), dtype=torch.bfloat16, device="cuda")
    yb = torch.zeros((3, 128), dtype=torch.float32, device="cuda")
    yc = torch.zeros((8, 256), dtype=torch.bfloat16, device="cuda")
    yd = torch.zeros((16, 640), dtype=torch.int32, device="cuda")
    ye = torch.zeros((8, 128), dtype=torch.float32, device="cuda")
    def stage(x, M, L, out, depends):
        return dict(x=x, M=M, K=L["K"], depends=depends,
                    linears=[dict(packed=L["packed"], w_scale=L["beta_d"], out=out, N=L["N"], out_dtype=L["dt"])])
    stages = [stage(dev_bf16(xa), 8, A, ya, 0), stage(dev_bf16(xb), 3, B, yb, 0),
              stage(ya, 8, C, yc, 1), stage(dev_bf16(xd), 16, D, yd, 0),
              stage(yc, 8, E_, ye, 1)]
    keep = [s["x"] for s in stages]
    prog = vla.compile_program(stages)
    for _ in range(2):
        vla.vla_program_run(prog)
    torch.cuda.synchronize()
    ra = oracle.ternary_linear(xa, A["w"], A["beta"])
    rb = oracle.ternary_linear(xb, B["w"], B["beta"])
    rc = oracle.ternary_linear(ra["ybf16"], C["w"], C["beta"])
    rd = oracle.ternary_linear(xd, D["w"], D["beta"])
    re_ = oracle.ternary_linear(rc["ybf16"], E_["w"], E_["beta"])
    assert np.array_equal(bits(ya), ra["ybf16"])
    assert np.array_equal(yb.cpu().numpy().view(np.uint32), rb["y32"].view(np.uint32))
    assert np.array_equal(bits(yc), rc["ybf16"])
    assert np.array_equal(yd.cpu().numpy(), rd["acc"])
    assert np.array_equal(ye.cpu().numpy().view(np.uint32), re_["y32"].view(np.uint32))


@pytest.mark.parametrize("mset", [(8, 3, 1, 5), (8, 16, 3, 1)])
def test_team_and_fifteen_way_stages_alternate(vla, oracle, mset):
    """Three dependent phases of 37 independent stages each, so that every stage's group is ~4 CTAs: phase A
    (K=256, N=1024: 8 granules per CTA -> the kernel's three-team mode, ring wraps twice), phase B (K=1024, N=128: one
    granule per CTA -> 15-way k split), phase C (K=128, N=1024: team mode again).  Every CTA therefore switches mode
    twice with the weight ring running across the switches; mset with a 16 selects the M <= 16 kernel variant
    (4 ring slots, B fragments of tokens 8-15 in shared memory), without it the M <= 8 variant (6 slots).
    Every output of every phase is compared with the oracle (bf16 chain, last phase fp32 / bf16 / int32)."""
    S = 37
    def lin(N, K, seed):
        w = synth.ternary_weights(N, K, 0.35, seed)
        beta = synth.weight_scale(seed + 1)
        return dict(w=w, beta=beta, packed=vla.pack_weights(dev(w)), beta_d=dev(np.array([beta], np.float32)), N=N, K=K)
    xs, A, B, C, ya, yb, yc, stages = [], [], [], [], [], [], [], []
    for i in range(S):
        M = mset[i % 4]
        xs.append(synth.activations(M, 256, 100 + i, outlier_frac=0.01))
        A.append(lin(1024, 256, 1000 + 3 * i)); B.append(lin(128, 1024, 2000 + 3 * i)); C.append(lin(1024, 128, 3000 + 3 * i))
        ya.append(torch.zeros((M, 1024), dtype=torch.bfloat16, device="cuda"))
        yb.append(torch.zeros((M, 128), dtype=torch.bfloat16, device="cuda"))
        yc.append(torch.full((M, 1024), -7, dtype=_TDT[i % 3], device="cuda"))
    def stage(x, M, L, out, depends, dt):
        return dict(x=x, M=M, K=L["K"], depends=depends,
                    linears=[dict(packed=L["packed"], w_scale=L["beta_d"], out=out, N=L["N"], out_dtype=dt)])
    xin = [dev_bf16(x) for x in xs]
    for i in range(S): stages.append(stage(xin[i], mset[i % 4], A[i], ya[i], 0, 1))
    for i in range(S): stages.append(stage(ya[i], mset[i % 4], B[i], yb[i], 1 if i == 0 else 0, 1))
    for i in range(S): stages.append(stage(yb[i], mset[i % 4], C[i], yc[i], 1 if i == 0 else 0, i % 3))
    prog = vla.compile_program(stages)
    for _ in range(3):
        vla.vla_program_run(prog)
    torch.cuda.synchronize()
    for i in range(S):
        ra = oracle.ternary_linear(xs[i], A[i]["w"], A[i]["beta"])
        rb = oracle.ternary_linear(ra["ybf16"], B[i]["w"], B[i]["beta"])
        rc = oracle.ternary_linear(rb["ybf16"], C[i]["w"], C[i]["beta"])
        assert np.array_equal(bits(ya[i]), ra["ybf16"]), "phase A stage %d" % i
        assert np.array_equal(bits(yb[i]), rb["ybf16"]), "phase B stage %d" % i
        if i % 3 == 2:
            assert np.array_equal(yc[i].cpu().numpy(), rc["acc"]), "phase C stage %d" % i
        elif i % 3 == 0:
            assert np.array_equal(yc[i].cpu().numpy().view(np.uint32), rc["y32"].view(np.uint32)), "phase C stage %d" % i
        else:
            assert np.array_equal(bits(yc[i]), rc["ybf16"]), "phase C stage %d" % i


def _guarded(shape, dtype, fill):
    """tensor view with 4 KiB of sentinel bytes on both sides (a hand-made out-of-bounds-write detector)"""
    n = int(np.prod(shape)) * torch.empty((), dtype=dtype).element_size()
    raw = torch.full((n + 8192,), 0xA5, dtype=torch.uint8, device="cuda")
    view = raw[4096:4096 + n].view(dtype).view(*shape)
    view.fill_(fill)
    return raw, view


def _guards_intact(raw):
    r = raw.cpu().numpy()
    return bool((r[:4096] == 0xA5).all() and (r[-4096:] == 0xA5).all())


def test_guard_bands_and_repeatability(vla, oracle):
    """No kernel writes outside its outputs (sentinels around every output, xq and alpha buffer survive), and 200
    back-to-back replays of a program with cross-CTA flags give the same bits every time (ragged shapes, M = 5 / 13)."""
    M, K = 5, 384
    x_bits = synth.activations(M, K, 321, outlier_frac=0.01)
    specs = [(128, 1), (384, 0), (256, 2)]
    raws, lins, refs = [], [], []
    for i, (N, dt) in enumerate(specs):
        w = synth.ternary_weights(N, K, 0.35, 700 + i)
        beta = synth.weight_scale(710 + i)
        raw, out = _guarded((M, N), _TDT[dt], 0)
        raws.append(raw)
        lins.append(dict(packed=vla.pack_weights(dev(w)), w_scale=dev(np.array([beta], np.float32)), out=out, N=N, out_dtype=dt))
        refs.append((oracle.ternary_linear(x_bits, w, beta), dt, out))
    rq, xq = _guarded((M, K), torch.int8, 0)
    rs, xs = _guarded((M,), torch.float32, 0)
    raws += [rq, rs]
    # second phase: M = 13 reads the bf16 output of the first linear (N = 128 -> K = 128)
    M2 = 13
    x2_bits = synth.activations(M2, 128, 322)
    w2 = synth.ternary_weights(640, 128, 0.35, 720)
    b2 = synth.weight_scale(721)
    raw2, out2 = _guarded((M2, 640), torch.bfloat16, 0)
    raws.append(raw2)
    stages = [dict(x=dev_bf16(x_bits), M=M, K=K, depends=0, linears=lins, xq_opt=xq, x_scale_opt=xs),
              dict(x=dev_bf16(x2_bits), M=M2, K=128, depends=1,
                   linears=[dict(packed=vla.pack_weights(dev(w2)), w_scale=dev(np.array([b2], np.float32)), out=out2, N=640, out_dtype=1)])]
    keep = [s["x"] for s in stages]
    prog = vla.compile_program(stages)
    g = torch.cuda.CUDAGraph()
    vla.vla_program_run(prog)
    torch.cuda.synchronize()
    with torch.cuda.graph(g):
        for _ in range(20):
            vla.vla_program_run(prog)
    first = None
    for rep in range(10):                                     # 200 runs
        g.replay()
        torch.cuda.synchronize()
        snap = [o.clone() for (_, _, o) in refs] + [out2.clone()]
        if first is None:
            first = snap
        else:
            assert all(torch.equal(a.view(torch.uint8), b.view(torch.uint8)) for a, b in zip(first, snap)), "run-to-run difference"
    for ref, dt, out in refs:
        if dt == 2:
            assert np.array_equal(out.cpu().numpy(), ref["acc"])
        elif dt == 0:
            assert np.array_equal(out.cpu().numpy().view(np.uint32), ref["y32"].view(np.uint32))
        else:
            assert np.array_equal(bits(out), ref["ybf16"])
    assert np.array_equal(xq.cpu().numpy(), refs[0][0]["a"])
    assert np.array_equal(bits(out2), oracle.ternary_linear(x2_bits, w2, b2)["ybf16"])
    assert all(_guards_intact(r) for r in raws), "a kernel wrote outside its buffer"


def test_program_run_host_sync_and_async_pipeline(vla, oracle):
    """vla_program_run_host (synchronous) and vla_program_run_host_async on two buffer sets / two streams (the serving loop
    of bench.py's end-to-end leg): pinned host x -> device -> program -> pinned host y, every output vs the oracle."""
    sets = []
    for b in range(2):
        pts = [make_point(vla, M, K, N, 9800 + 10 * b + i, vla.VLA_BF16) for i, (M, K, N) in enumerate([(8, 2560, 640), (16, 640, 256)])]
        hx = [torch.empty(p["x"].shape, dtype=torch.bfloat16).pin_memory() for p in pts]
        hy = [torch.zeros(p["out"].shape, dtype=torch.bfloat16).pin_memory() for p in pts]
        for h, p in zip(hx, pts):
            h.copy_(p["x"].cpu())
            p["x"].zero_()                                   # the device copy must come from the host buffer
        prog = vla.compile_program([stage_of(p) for p in pts])
        cin = vla.make_copies([(h, p["x"]) for h, p in zip(hx, pts)])
        cout = vla.make_copies([(h, p["out"]) for h, p in zip(hy, pts)])
        sets.append(dict(pts=pts, hx=hx, hy=hy, prog=prog, cin=cin, cout=cout, stream=torch.cuda.Stream()))

    def check(s):
        for h, p in zip(s["hy"], s["pts"]):
            ref = oracle.ternary_linear(p["x_bits"], p["w"], p["beta"])
            assert np.array_equal(h.view(torch.int16).numpy().view(np.uint16), ref["ybf16"])
            h.zero_()

    vla.vla_program_run_host(sets[0]["prog"], sets[0]["cin"], sets[0]["cout"])          # synchronous: results are there
    check(sets[0])
    torch.cuda.synchronize()
    for rep in range(3):                                     # asynchronous, alternating sets and streams
        for s in sets:
            vla.vla_program_run_host_async(s["prog"], s["cin"], s["cout"], s["stream"])
        for s in sets:
            s["stream"].synchronize()
            check(s)
    for s in sets:
        vla.vla_program_release(s["prog"])
