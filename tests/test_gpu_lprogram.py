"""GPU parity tests (-m gpu) of LARGE programs (vla_program_build / vla_program_run with M > 16 tokens per stage): the
persistent tcgen05 kernel of csrc/gemm_lprog.cu -- activation quant fused into the launch (rows quantised cooperatively
by the CTAs, grid-wide counters), stages chained without leaving the kernel -- against the CPU oracle.  Every output is
compared element by element and is bit-identical (canonical operation order, R1, R6).
"""
import numpy as np
import pytest
import torch

from paper_2606_08094_b200 import synth
from test_gpu_program import bits, check_point, dev, dev_bf16, make_point, oracle_stack, stage_of, vla  # noqa: F401

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("M,K,N", [(17, 128, 128), (32, 256, 256), (100, 640, 384), (200, 2560, 640), (544, 2560, 2560),
                                   (545, 6912, 2560), (1000, 2560, 6912), (2500, 1024, 256), (333, 8192, 128)])
@pytest.mark.parametrize("dtype", [0, 1, 2])
def test_single_stage_large_program(vla, oracle, M, K, N, dtype):
    """one linear per program: token tiles of 32..256, one and two k blocks per pipeline stage, ragged M, one to several
    waves of tiles, 1..28 rows per CTA in the fused quantiser (several rounds), every output type; also the optional
    xq / alpha outputs"""
    p = make_point(vla, M, K, N, 9100 + M + K + N, dtype, want_xq=True)
    prog = vla.compile_program([stage_of(p)])
    vla.vla_program_run(prog)
    torch.cuda.synchronize()
    check_point(vla, oracle, p)
    vla.vla_program_release(prog)


def test_grouped_stage_mixed_dtypes_scratch_activations(vla, oracle):
    """one stage, three linears with their own beta and output type (Eq. 4's per-output-group scales), ragged M=545,
    quantised activations kept in the program's scratch (no xq_opt)"""
    M, K = 545, 2560
    x = synth.activations(M, K, 9301, outlier_frac=0.01)
    lins, refs = [], []
    for j, (N, dt) in enumerate([(2560, vla.VLA_BF16), (640, vla.VLA_F32), (640, vla.VLA_I32)]):
        p = make_point(vla, M, K, N, 9310 + j, dt)
        p["x_bits"], p["x"] = x, None
        lins.append(p)
    xd = dev_bf16(x)
    stage = dict(x=xd, M=M, K=K, depends=0,
                 linears=[dict(packed=p["packed"], w_scale=p["beta_d"], out=p["out"], N=p["N"], out_dtype=p["dtype"]) for p in lins])
    prog = vla.compile_program([stage])
    for rep in range(3):
        for p in lins:
            p["out"].fill_(-5)
        vla.vla_program_run(prog)
        torch.cuda.synchronize()
        for p in lins:
            check_point(vla, oracle, p)
    vla.vla_program_release(prog)


def test_independent_stages_alternate_scratch_and_rerun(vla, oracle):
    """seven independent stages of different M, K, N in one launch (the two scratch pairs alternate; the token tile and the
    reserved X tile differ per stage), run three times and once from a CUDA graph: the counters reset themselves"""
    shapes = [(64, 2560, 640), (544, 640, 1280), (200, 6912, 256), (17, 256, 128), (1024, 1280, 384), (96, 8192, 256),
              (300, 384, 2560)]
    pts = [make_point(vla, M, K, N, 9400 + i, [1, 0, 2][i % 3]) for i, (M, K, N) in enumerate(shapes)]
    prog = vla.compile_program([stage_of(p) for p in pts])
    for rep in range(3):
        for p in pts:
            p["out"].fill_(-3)
        vla.vla_program_run(prog)
        torch.cuda.synchronize()
        for p in pts:
            check_point(vla, oracle, p)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        vla.vla_program_run(prog)
        vla.vla_program_run(prog)
    for p in pts:
        p["out"].fill_(-3)
    g.replay()
    torch.cuda.synchronize()
    for p in pts:
        check_point(vla, oracle, p)
    vla.vla_program_release(prog)


@pytest.mark.parametrize("M,K", [(544, 512), (544, 384), (1100, 512), (100, 256)])
def test_long_program_work_tiles_and_round_robin(vla, oracle, M, K):
    """A program long enough for the work-minimising token tiles and the tile round robin across stages (20 independent
    or 40 stages, N alternating 3840 / 2560 / 1280): M=544 -> TN = 192, A operand in tensor memory with 192-column accumulators, two
    k blocks per stage (K=512) or one (K=384: odd number of k blocks); M=1100 -> TN = 256, A operand in shared memory;
    M=100 -> TN = 112, 128-column accumulators.  Most stages have fewer tiles than SMs, so each starts on the CTAs the
    previous one left idle.  Every output vs the oracle, twice."""
    Ns = [3840, 2560, 1280]                                  # 30 / 20 / 10 channel tiles: > 4 x 148 tiles in all = "long"
    n_st = 20 if M >= 544 else 40
    pts = [make_point(vla, M, K, Ns[i % 3], 9900 + i, [0, 1, 2][i % 3], want_xq=(i % 5 == 0)) for i in range(n_st)]
    prog = vla.compile_program([stage_of(p) for p in pts])
    for rep in range(2):
        for p in pts:
            p["out"].fill_(-3)
        vla.vla_program_run(prog)
        torch.cuda.synchronize()
        for p in pts:
            check_point(vla, oracle, p)
    vla.vla_program_release(prog)


def test_random_large_programs_equal_single_calls(vla):
    """Seeded random large programs (1..12 stages, M from 17 to 2048, K and N from the small shapes, ~30 % of the stages
    reading the previous stage's bf16 output) run three times: outputs are deterministic and bit-identical to one
    vla_ternary_linear call per stage on the same inputs (which test_gpu_parity.py checks against the oracle)."""
    rng = np.random.default_rng(20260608)
    for trial in range(14):
        M = int(rng.choice([17, 33, 64, 100, 200, 544, 545, 1000, 1100, 2048]))
        stages = []
        for i in range(int(rng.integers(1, 13))):
            K = int(rng.choice([128, 256, 384, 512, 640, 1280]))
            N = int(rng.choice([128, 256, 384, 640, 1280]))
            packed = vla.pack_weights(dev(synth.ternary_weights(N, K, 0.35, int(rng.integers(1 << 30)))))
            beta = dev(np.array([synth.weight_scale(int(rng.integers(1 << 30)))], np.float32))
            chained = i > 0 and rng.random() < 0.3 and stages[-1]["linears"][0]["N"] == K
            x = stages[-1]["linears"][0]["out"] if chained else dev_bf16(synth.activations(M, K, int(rng.integers(1 << 30))))
            out = torch.zeros((M, N), dtype=torch.bfloat16, device="cuda")
            stages.append(dict(x=x, M=M, K=K, depends=1 if chained else 0,
                               linears=[dict(packed=packed, w_scale=beta, out=out, N=N, out_dtype=vla.VLA_BF16)]))
        prog = vla.compile_program(stages)
        vla.vla_program_run(prog)
        torch.cuda.synchronize()
        first = [st["linears"][0]["out"].clone() for st in stages]
        for rep in range(2):
            vla.vla_program_run(prog)
        torch.cuda.synchronize()
        for st, ref in zip(stages, first):
            lin = st["linears"][0]
            assert torch.equal(lin["out"], ref), "trial %d: output changed between runs" % trial
            nb = vla.vla_ternary_workspace_bytes(M, lin["N"], st["K"])
            ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
            single = torch.empty_like(ref)
            vla.vla_ternary_linear(lin["packed"], lin["w_scale"], st["x"], M, lin["N"], st["K"], single, vla.VLA_BF16,
                                   vla.VLA_PATH_AUTO, None, None, ws, nb)
            torch.cuda.synchronize()
            assert torch.equal(single, ref), "trial %d: M=%d K=%d N=%d differs from the single call" % (trial, M, st["K"], lin["N"])
        vla.vla_program_release(prog)


@pytest.mark.parametrize("M", [512, 1024])
def test_wide_stages_equal_single_call(vla, M):
    """Twelve independent (8192 -> 8192) stages on the same x with their own weights: 16 KB rows (the quantiser's row buffer
    takes one chunk of 2-3 rows at a time, not double-buffered), 64 k blocks per tile, the packed-weight ring running far
    ahead across stage boundaries.  (A 3-deep weight ring failed exactly here: with an odd depth a decode group's parity
    wait falls through -- the ring depth is even now.)  Three runs, every stage bit-identical to one
    vla_ternary_linear call with the same weights."""
    K = N = 8192
    n_st = 12
    x = dev_bf16(synth.activations(M, K, 77001))
    w0 = vla.pack_weights(dev(synth.ternary_weights(N, K, 0.35, 77002)))
    ring = w0.unsqueeze(0).repeat(n_st, 1).contiguous()
    for c in range(1, n_st):                                  # distinct weights per stage: rotate the packed channel blocks
        ring[c] = torch.roll(w0, shifts=c * (K // 4) * 128)
    beta = dev(np.array([0.05], np.float32))
    outs = [torch.zeros((M, N), dtype=torch.bfloat16, device="cuda") for _ in range(n_st)]
    stages = [dict(x=x, M=M, K=K, depends=0, linears=[dict(packed=ring[c], w_scale=beta, out=outs[c], N=N, out_dtype=vla.VLA_BF16)])
              for c in range(n_st)]
    prog = vla.compile_program(stages)
    nb = vla.vla_ternary_workspace_bytes(M, N, K)
    ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
    single = torch.empty((M, N), dtype=torch.bfloat16, device="cuda")
    for rep in range(3):
        for o in outs:
            o.fill_(-3)
        vla.vla_program_run(prog)
        torch.cuda.synchronize()
        for c in (0, 1, 5, n_st - 1) if rep else range(n_st):
            vla.vla_ternary_linear(ring[c], beta, x, M, N, K, single, vla.VLA_BF16, vla.VLA_PATH_AUTO, None, None, ws, nb)
            torch.cuda.synchronize()
            assert torch.equal(outs[c], single), "run %d stage %d differs from the single call" % (rep, c)
    assert not torch.equal(outs[0], outs[1])
    vla.vla_program_release(prog)


def test_chained_stages_with_several_quantiser_chunks(vla):
    """M = 2048 rows of K = 2560 are 14 rows per CTA: the fused quantiser takes them in several double-buffered chunks, and
    in a DEPENDENT chain the first chunk of a stage may only be loaded once the previous stage is stored everywhere (no
    prefetch across the stage boundary, proxy fence before the copies).  Four chained stages + one independent stage in
    between, three runs, bit-identical to the same chain of single vla_ternary_linear calls."""
    M = 2048
    shapes = [(2560, 2560, 1), (2560, 2560, 1), (2560, 1280, 0), (2560, 2560, 1), (2560, 640, 1)]   # (K, N, reads the previous output)
    x0 = dev_bf16(synth.activations(M, 2560, 88001))
    x_ind = dev_bf16(synth.activations(M, 2560, 88002))
    packed = [vla.pack_weights(dev(synth.ternary_weights(N, K, 0.35, 88010 + i))) for i, (K, N, _) in enumerate(shapes)]
    beta = dev(np.array([0.03], np.float32))
    outs = [torch.zeros((M, N), dtype=torch.bfloat16, device="cuda") for (_, N, _) in shapes]
    stages, xin = [], []
    last_chain = None                                         # index of the last stage of the chain so far
    for i, (K, N, dep) in enumerate(shapes):
        if i == 0:
            x, d = x0, 0
        elif dep:
            x, d = outs[last_chain], i - last_chain
        else:
            x, d = x_ind, 0
        if dep or i == 0:
            last_chain = i
        xin.append(x)
        stages.append(dict(x=x, M=M, K=K, depends=d, linears=[dict(packed=packed[i], w_scale=beta, out=outs[i], N=N, out_dtype=vla.VLA_BF16)]))
    prog = vla.compile_program(stages)
    got = None
    for rep in range(3):
        for o in outs:
            o.fill_(-3)
        vla.vla_program_run(prog)
        torch.cuda.synchronize()
        if got is None:
            got = [o.clone() for o in outs]
        else:
            for a, b in zip(outs, got):
                assert torch.equal(a, b), "run %d differs from the first" % rep
    refs = []
    for i, (K, N, dep) in enumerate(shapes):
        nb = vla.vla_ternary_workspace_bytes(M, N, K)
        ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
        ref = torch.empty((M, N), dtype=torch.bfloat16, device="cuda")
        if i == 0:
            x = x0
        elif dep:
            x = refs[max(j for j in range(i) if shapes[j][2] or j == 0)]
        else:
            x = x_ind
        vla.vla_ternary_linear(packed[i], beta, x, M, N, K, ref, vla.VLA_BF16, vla.VLA_PATH_AUTO, None, None, ws, nb)
        torch.cuda.synchronize()
        refs.append(ref)
        assert torch.equal(got[i], ref), "stage %d differs from the chain of single calls" % i
    vla.vla_program_release(prog)


def test_chained_stack_m544_one_launch(vla, oracle):
    """configs[3] at M=544 as ONE launch: 3 full-size layers = 12 dependent stages (q|k|v as one N=3840 group, gate|up as
    N=13824), quantisation fused, free-running; every intermediate of every layer bit-identical to the oracle's chain.
    Run twice (stale activations of the first run are still in the scratch and in L2 during the second)."""
    from paper_2606_08094_b200.stack import Stack
    layers, M = 3, synth.PREFILL_M
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
                st.out[l][n].zero_()


@pytest.mark.parametrize("blocks", [2, 3])
def test_chained_stack_as_interleaved_row_blocks(vla, oracle, blocks):
    """depends = d: the M=544 chain as `blocks` independent chains over row blocks of the batch, their stages interleaved in
    one launch (stage s waits only for the stages up to s - blocks).  2 full-size layers, every intermediate bit-identical to
    the oracle's chain, twice."""
    from paper_2606_08094_b200.stack import Stack
    layers, M = 2, synth.PREFILL_M
    weights = [synth.stack_layer(l) for l in range(layers)]
    x = synth.stack_input(M)
    st = Stack(layers, M, weights=weights)
    st.set_input(x)
    st.compile(blocks)
    ref = oracle_stack(oracle, weights, x)
    for rep in range(2):
        st.run_program()
        torch.cuda.synchronize()
        for l in range(layers):
            for n in ref[l]:
                assert np.array_equal(bits(st.out[l][n]), ref[l][n]), "layer %d %s differs (rep %d)" % (l, n, rep)
                st.out[l][n].zero_()


def test_chained_large_program_changing_inputs(vla, oracle):
    """a dependent pair (stage 1 reads stage 0's bf16 output) re-run with NEW inputs in the same buffers: a stale row in an
    SM's L1 or a stale alpha would show"""
    M, K, N1, N2 = 130, 640, 1280, 256
    a = make_point(vla, M, K, N1, 9500, vla.VLA_BF16)
    b = make_point(vla, M, N1, N2, 9510, vla.VLA_F32)
    st0 = stage_of(a)
    st1 = dict(stage_of(b), x=a["out"], depends=1)
    prog = vla.compile_program([st0, st1])
    for rep in range(3):
        x = synth.activations(M, K, 9520 + rep, outlier_frac=0.01)
        a["x"].copy_(dev_bf16(x))
        vla.vla_program_run(prog)
        torch.cuda.synchronize()
        r0 = oracle.ternary_linear(x, a["w"], a["beta"])
        assert np.array_equal(bits(a["out"]), r0["ybf16"])
        r1 = oracle.ternary_linear(r0["ybf16"], b["w"], b["beta"])
        assert np.array_equal(b["out"].cpu().numpy().view(np.uint32), r1["y32"].view(np.uint32))
    vla.vla_program_release(prog)


def test_large_program_guard_bands(vla, oracle):
    """nothing is written outside [M,N] / [M,K] / [M]: outputs and the optional xq / alpha live inside guarded buffers"""
    M, K, N = 77, 384, 256
    p = make_point(vla, M, K, N, 9600, vla.VLA_F32)
    G = 512
    out = torch.full((M * N + 2 * G,), 1234.5, dtype=torch.float32, device="cuda")
    xq = torch.full((M * K + 2 * G,), 55, dtype=torch.int8, device="cuda")
    xs = torch.full((M + 2 * G,), -9.0, dtype=torch.float32, device="cuda")
    p["out"] = out[G:G + M * N].view(M, N)
    p["xq"] = xq[G:G + M * K].view(M, K)
    p["xs"] = xs[G:G + M]
    prog = vla.compile_program([stage_of(p)])
    vla.vla_program_run(prog)
    torch.cuda.synchronize()
    check_point(vla, oracle, p)
    for t, v in ((out, 1234.5), (xq, 55), (xs, -9.0)):
        n = t.numel()
        inner = {id(out): M * N, id(xq): M * K, id(xs): M}[id(t)]
        assert bool((t[:G] == v).all()) and bool((t[G + inner:n] == v).all())
    vla.vla_program_release(prog)


def test_large_program_errors(vla):
    small = make_point(vla, 8, 256, 256, 5, vla.VLA_BF16)
    large = make_point(vla, 64, 256, 256, 6, vla.VLA_BF16)
    assert vla.vla_program_bytes([stage_of(small), stage_of(large)]) == 0          # one kind per program
    assert vla.vla_program_bytes([dict(stage_of(large), M=32769)]) == 0
    assert vla.vla_program_bytes([dict(stage_of(large), K=8192 + 128)]) == 0
    nine = stage_of(large)
    nine["linears"] = nine["linears"] * 9
    assert vla.vla_program_bytes([nine]) == 0                                      # at most 8 linears per large stage
    assert vla.vla_program_bytes([stage_of(large)]) > 0
    assert vla.vla_program_bytes([stage_of(large), dict(stage_of(large), depends=2)]) == 0      # depends <= stage index
    assert vla.vla_program_bytes([stage_of(large), stage_of(large), dict(stage_of(large), depends=2)]) > 0
