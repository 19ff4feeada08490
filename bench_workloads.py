"""Extra bench.py workloads: BASELINE.json configs[3] (30-layer chained stack) and configs[4] (roofline sweep).

Imported by bench.py only.  Timing protocol as in bench.py: CUDA graphs, CUDA events on the launching stream,
cold weights (the stack is 521 MB >> L2; the sweep rotates through a ring of packed copies > 2 x L2).
"""
import json
import os
import time

import numpy as np


def _events(torch):
    return torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)


def _time(torch, fn, reps):
    fn()
    torch.cuda.synchronize()
    e0, e1 = _events(torch)
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    e1.synchronize()
    return e0.elapsed_time(e1) * 1e-3 / reps


# ----------------------------------------------------------------------------- configs[3]
def run_stack(args, pk, clock_sampler):
    """30 decoder layers, q/k/v/o/gate/up/down ternary linears + their activation quant, chained; M=544 (one quant
    kernel + one grouped tcgen05 GEMM launch per stage, CUDA graph + PDL) then M=8 (ONE persistent program launch)."""
    import torch
    from paper_2606_08094_b200 import binding as vla, synth
    from paper_2606_08094_b200.stack import Stack
    layers = synth.STACK_LAYERS
    out = {}
    sampler = clock_sampler
    sampler.start()
    for M in (synth.PREFILL_M, 8):
        st = Stack(layers, M)
        st.set_input(synth.stack_input(M))
        n0 = vla.vla_launch_count()
        if M <= 16:
            st.compile()
            fn = st.run_program
            fn()
            launches = vla.vla_launch_count() - n0
        else:
            st.alloc_call_workspace()
            st.run_stack_calls()
            torch.cuda.synchronize()
            n0 = vla.vla_launch_count()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g):
                st.run_stack_calls()
            launches = vla.vla_launch_count() - n0
            fn = g.replay
        for _ in range(max(3, args.warmup // 4)):
            fn()
        sec = _time(torch, fn, max(3, min(args.steps, 50)))
        ops = 2.0 * M * sum(K * N for (_, K, N) in synth.STACK_LINEARS) * layers
        wbytes = float(st.packed_bytes)
        t_roof = max(wbytes / (pk["hbm_gbs"] * 1e9), ops / (pk["bf16_tflops"] * 2e12))
        out["M%d" % M] = {"us": sec * 1e6, "us_per_layer": sec * 1e6 / layers, "launches": launches,
                          "weight_GBs": wbytes / sec / 1e9, "TOPS": ops / sec / 1e12, "roofline_frac": t_roof / sec,
                          "route": "one persistent program launch" if M <= 16 else "act_quant + one grouped tcgen05 launch per stage, CUDA graph + PDL"}
        del st
        torch.cuda.empty_cache()
    clocks = sampler.stop()
    m8 = out["M8"]
    line = {
        "metric": "ternary_stack_weight_stream_gbs", "value": m8["weight_GBs"], "unit": "GB/s", "n_gpus": 1,
        "steps": max(3, min(args.steps, 50)), "warmup": max(3, args.warmup // 4), "ms_per_step": m8["us"] * 1e-3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int8*ternary->int32",
        "data": "synthetic",
        "config": {"workload": "configs[3] 30-layer stack (hidden 2560, 20q/5kv x128, FFN 6912), linears + quant chained; "
                               "value is the M=8 pass", "cold_weights": "521 MB packed per pass (>> L2)"},
        "clocks": clocks, "gpu_launches": m8["launches"], "stack": out,
        "roofline": {"bound": "hbm", "achieved": m8["weight_GBs"], "peak": pk["hbm_gbs"], "unit": "GB/s",
                     "frac": m8["weight_GBs"] / pk["hbm_gbs"], "traffic": None, "kernel": "program_kernel"},
    }
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------- configs[4]
def run_sweep(args, pk, clock_sampler, int8_probe_tops):
    """M in {1..4096} x 4 shapes x zero fraction x activation distribution, fused quant, fp32 out: TOPS, GB/s and
    roofline fraction per point (single vla_ternary_linear calls in a CUDA graph over a cold ring); for M <= 16 also
    the streaming regime (a ring-full of the same linear as independent stages of one persistent program)."""
    import torch
    from paper_2606_08094_b200 import binding as vla, synth
    dev = torch.device("cuda", 0)
    l2 = torch.cuda.get_device_properties(dev).L2_cache_size
    peak_i8 = pk["bf16_tflops"] * 2.0
    Ms = synth.SWEEP_M if not args.sweep_m else [int(m) for m in args.sweep_m.split(",")]
    zfs = range(len(synth.SWEEP_ZERO_FRAC)) if not args.quick else [1]
    dists = range(len(synth.SWEEP_DISTS)) if not args.quick else [0]
    pts = []
    sampler = clock_sampler
    sampler.start()
    for si, (K, N) in enumerate(synth.SWEEP_SHAPES):
        copies = max(2, -(-2 * l2 // (N * K // 4)))
        Mmax = max(Ms)
        for zf in zfs:
            w = synth.ternary_weights(N, K, synth.SWEEP_ZERO_FRAC[zf], 4000 + 10 * si + zf)
            packed1 = vla.pack_weights(torch.from_numpy(w).to(dev))
            ring = packed1.unsqueeze(0).repeat(copies, 1).contiguous()
            del w, packed1
            beta = torch.tensor([0.05], dtype=torch.float32, device=dev)
            for di in dists:
                xb = synth.activations(Mmax, K, 504000 + 10 * si + di, dist=synth.SWEEP_DISTS[di])
                x_all = torch.from_numpy(xb.view(np.int16)).to(dev).view(torch.bfloat16)
                for M in Ms:
                    x = x_all[:M].contiguous()
                    out = torch.empty((M, N), dtype=torch.float32, device=dev)
                    xq = torch.empty((M, K), dtype=torch.int8, device=dev)
                    xs = torch.empty((M,), dtype=torch.float32, device=dev)
                    nb = vla.vla_ternary_workspace_bytes(M, N, K)
                    ws = torch.empty(nb, dtype=torch.uint8, device=dev)
                    ncall = min(copies, 32)

                    def calls():
                        for c in range(ncall):
                            vla.vla_ternary_linear(ring[c], beta, x, M, N, K, out, vla.VLA_F32, vla.VLA_PATH_AUTO, xq, xs, ws, nb)
                    calls()
                    torch.cuda.synchronize()
                    g = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(g):
                        calls()
                    sec = _time(torch, g.replay, 3 if M >= 1024 else 10) / ncall
                    by = N * K // 4 + 4 + 2 * M * K + 4 * M * N
                    op = 2.0 * M * N * K
                    t_roof = max(by / (pk["hbm_gbs"] * 1e9), op / (peak_i8 * 1e12))
                    p = {"M": M, "K": K, "N": N, "zero_frac": synth.SWEEP_ZERO_FRAC[zf], "dist": synth.SWEEP_DISTS[di],
                         "us": sec * 1e6, "TOPS": op / sec / 1e12, "GBs": by / sec / 1e9, "roofline_frac": t_roof / sec,
                         "bound": "hbm" if by / (pk["hbm_gbs"] * 1e9) > op / (peak_i8 * 1e12) else "tensor",
                         "path": int(vla.vla_ternary_auto_path(M, N, K))}
                    if M <= 16 and zf == list(zfs)[0] and di == list(dists)[0]:
                        nst = min(copies, 128)
                        outs = [torch.empty((M, N), dtype=torch.float32, device=dev) for _ in range(nst)]
                        stages = [dict(x=x, M=M, K=K, depends=0,
                                       linears=[dict(packed=ring[c], w_scale=beta, out=outs[c], N=N, out_dtype=vla.VLA_F32)])
                                  for c in range(nst)]
                        prog = vla.compile_program(stages, dev)
                        secp = _time(torch, lambda: vla.vla_program_run(prog), 10) / nst
                        p["stream_us"] = secp * 1e6
                        p["stream_GBs"] = by / secp / 1e9
                        p["stream_roofline_frac"] = (by / (pk["hbm_gbs"] * 1e9)) / secp
                        vla.vla_program_release(prog)
                        del prog, outs
                    pts.append(p)
                    del g
                del x_all
            del ring
            torch.cuda.empty_cache()
    # NEXT-3: the paper's dp4a -> tensor-core comparison (4.0-4.6x end to end at S=8 on RTX 3060 / AGX Orin,
    # PAPER.md line 130) restated kernel to kernel on this B200 at M=8: same packed weights, same pre-quantised
    # activations, VLA_PATH_SMALL_ALU (dp4a on the integer ALUs) vs VLA_PATH_SMALL_TC (IMMA), cold ring, CUDA graph.
    compare = []
    for si, (K, N) in enumerate(synth.MODEL_SHAPES):
        M = 8
        copies = max(2, -(-2 * l2 // (N * K // 4)))
        w = synth.ternary_weights(N, K, 0.35, 4900 + si)
        packed1 = vla.pack_weights(torch.from_numpy(w).to(dev))
        ring = packed1.unsqueeze(0).repeat(copies, 1).contiguous()
        del w, packed1
        beta = torch.tensor([0.05], dtype=torch.float32, device=dev)
        xq = torch.randint(-127, 128, (M, K), dtype=torch.int8, device=dev)
        xs = torch.rand(M, device=dev) + 0.01
        out = torch.empty((M, N), dtype=torch.bfloat16, device=dev)
        row = {"M": M, "K": K, "N": N}
        for name, path in (("dp4a_us", vla.VLA_PATH_SMALL_ALU), ("imma_us", vla.VLA_PATH_SMALL_TC)):
            ncall = min(copies, 64)

            def calls():
                for c in range(ncall):
                    vla.vla_ternary_gemm(ring[c], beta, xq, xs, M, N, K, out, vla.VLA_BF16, path, None, 0)
            calls()
            torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g):
                calls()
            row[name] = _time(torch, g.replay, 10) / ncall * 1e6
            del g
        row["imma_over_dp4a"] = row["dp4a_us"] / row["imma_us"]
        compare.append(row)
        del ring
        torch.cuda.empty_cache()
    # Row a6 evidence for 16 < M <= 32: the IMMA kernel and the tcgen05 kernel, forced, on the same fused
    # vla_ternary_linear call over cold weights; "auto" is what VLA_PATH_AUTO resolves to.
    crossover = []
    for si, (K, N) in enumerate(list(synth.SWEEP_SHAPES) + [(2560, 640)]):
        copies = max(2, -(-2 * l2 // (N * K // 4)))
        w = synth.ternary_weights(N, K, 0.33, 4950 + si)
        packed1 = vla.pack_weights(torch.from_numpy(w).to(dev))
        ring = packed1.unsqueeze(0).repeat(copies, 1).contiguous()
        del w, packed1
        beta = torch.tensor([0.05], dtype=torch.float32, device=dev)
        xb = synth.activations(32, K, 505000 + si)
        x_all = torch.from_numpy(xb.view(np.int16)).to(dev).view(torch.bfloat16)
        for M in (17, 24, 32):
            x = x_all[:M].contiguous()
            out = torch.empty((M, N), dtype=torch.float32, device=dev)
            xq = torch.empty((M, K), dtype=torch.int8, device=dev)
            xs = torch.empty((M,), dtype=torch.float32, device=dev)
            row = {"M": M, "K": K, "N": N, "auto": int(vla.vla_ternary_auto_path(M, N, K))}
            for name, path in (("small_tc_us", vla.VLA_PATH_SMALL_TC), ("large_us", vla.VLA_PATH_LARGE)):
                ncall = min(copies, 32)

                def calls():
                    for c in range(ncall):
                        vla.vla_ternary_linear(ring[c], beta, x, M, N, K, out, vla.VLA_F32, path, xq, xs, None, 0)
                calls()
                torch.cuda.synchronize()
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g):
                    calls()
                row[name] = _time(torch, g.replay, 10) / ncall * 1e6
                del g
            crossover.append(row)
        del ring, x_all
        torch.cuda.empty_cache()
    clocks = sampler.stop()
    big = [p for p in pts if p["M"] >= 512]
    small = [p for p in pts if p["M"] <= 16]
    best_big = max(big, key=lambda p: p["roofline_frac"]) if big else None
    line = {
        "metric": "ternary GEMM TOPS & HBM GB/s vs M; fraction of INT8/HBM roofline (1 B200)",
        "value": best_big["TOPS"] if best_big else 0.0, "unit": "TOP/s", "n_gpus": 1, "steps": len(pts), "warmup": 1,
        "ms_per_step": None, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int8*ternary->int32", "data": "synthetic",
        "config": {"workload": "configs[4] roofline sweep, %d points, fused quant, fp32 out; value = best M>=512 point" % len(pts),
                   "cold_weights": "ring of packed copies > 2 x L2 per shape"},
        "clocks": clocks,
        "peaks": {"hbm_gbs": pk["hbm_gbs"], "int8_tops_bf16x2": peak_i8, "int8_tops_probe": int8_probe_tops,
                  "int8_tops_nominal": 4500.0},
        "summary": {
            "M>=512 roofline_frac min/median/max": [float(np.min([p["roofline_frac"] for p in big])),
                                                    float(np.median([p["roofline_frac"] for p in big])),
                                                    float(np.max([p["roofline_frac"] for p in big]))] if big else None,
            "M<=16 single-call roofline_frac median": float(np.median([p["roofline_frac"] for p in small])) if small else None,
            "M<=16 streaming roofline_frac median": float(np.median([p["stream_roofline_frac"] for p in small
                                                                     if "stream_roofline_frac" in p])) if small else None},
        "dp4a_vs_imma_M8": compare,
        "path_crossover_M17_32": crossover,
        "points": pts,
    }
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------- row a6: forced paths side by side (ncu target)
def run_dispatch(args, pk, clock_sampler):
    """Row a6 evidence: the kernels the dispatcher chooses between, forced, on the same pre-quantised inputs over cold
    packed weights -- dp4a (VLA_PATH_SMALL_ALU) vs IMMA (VLA_PATH_SMALL_TC) at M in {8, 16}, IMMA vs tcgen05
    (VLA_PATH_LARGE) at M in {17, 24, 32}.  Few eager launches per point (3 timed), so that an
    `ncu --metrics ... -k regex:gemm_` pass over this command stays short; profiles/r02_dispatch_ncu.md is that pass."""
    import torch
    from paper_2606_08094_b200 import binding as vla, synth
    dev = torch.device("cuda", 0)
    l2 = torch.cuda.get_device_properties(dev).L2_cache_size
    flush = torch.empty(2 * l2, dtype=torch.uint8, device=dev)
    rows = []
    clock_sampler.start()
    for si, (K, N) in enumerate(synth.MODEL_SHAPES):
        w = synth.ternary_weights(N, K, 0.35, 4900 + si)
        packed = vla.pack_weights(torch.from_numpy(w).to(dev))
        beta = torch.tensor([0.05], dtype=torch.float32, device=dev)
        for M, paths in ((8, ("SMALL_ALU", "SMALL_TC")), (16, ("SMALL_ALU", "SMALL_TC")),
                         (17, ("SMALL_TC", "LARGE")), (24, ("SMALL_TC", "LARGE")), (32, ("SMALL_TC", "LARGE"))):
            xq = torch.randint(-127, 128, (M, K), dtype=torch.int8, device=dev)
            xs = torch.rand(M, device=dev) + 0.01
            out = torch.empty((M, N), dtype=torch.bfloat16, device=dev)
            row = {"M": M, "K": K, "N": N, "auto": int(vla.vla_ternary_auto_path(M, N, K))}
            for name in paths:
                path = getattr(vla, "VLA_PATH_" + name)
                us = []
                for _ in range(4):                                  # first one is the warm-up
                    flush.fill_(1)                                   # weights leave L2
                    e0, e1 = _events(torch)
                    e0.record()
                    vla.vla_ternary_gemm(packed, beta, xq, xs, M, N, K, out, vla.VLA_BF16, path, None, 0)
                    e1.record()
                    e1.synchronize()
                    us.append(e0.elapsed_time(e1) * 1e3)
                row[name + "_us"] = float(np.median(us[1:]))
            rows.append(row)
        del packed
    clocks = clock_sampler.stop()
    print(json.dumps({"metric": "ternary GEMM TOPS & HBM GB/s vs M; fraction of INT8/HBM roofline (1 B200)",
                      "value": None, "unit": "us per forced-path launch (eager, cold weights, includes launch overhead)",
                      "n_gpus": 1, "steps": 3, "warmup": 1, "higher_is_better": False, "data": "synthetic",
                      "config": {"workload": "row a6 dispatch evidence: forced paths on the four model shapes"},
                      "clocks": clocks, "dispatch": rows}))
    return 0


# ----------------------------------------------------------------------------- the metric "vs M" (default bench.py line)
VS_M_SHAPES = [(2560, 2560), (2560, 640), (2560, 6912), (6912, 2560), (8192, 8192)]
VS_M_M = [1, 8, 16, 64, 512, 544, 1024, 4096]


def run_vs_m(pk, int8_probe_tops, Ms=None, shapes=None):
    """BASELINE.json's metric is "TOPS & HBM GB/s vs M; fraction of INT8/HBM roofline": the four model shapes and 8192^2
    at M in {1, 8, 16, 64, 512, 544, 1024, 4096}, fused quant (vla_ternary_linear, VLA_PATH_AUTO, fp32 out), every call
    of a CUDA graph on its own packed-weight copy of a ring larger than 2 x L2 (cold weights); beside it the program
    route (the ring as independent stages of one persistent launch: program_kernel for M <= 16, lprog_kernel with the
    quant fused for M > 16).  Returns (points, roofline_tensor) where roofline_tensor is the record of the dominant kernel
    of the M >= 512 half: lprog_kernel on the configs[2] prefill step (four model shapes, M = 544, Eq. 4 end to end), with
    gemm_large_kernel alone on pre-quantised activations nested under "gemm_only"."""
    import torch
    from paper_2606_08094_b200 import binding as vla, synth
    dev = torch.device("cuda", torch.cuda.current_device())
    l2 = torch.cuda.get_device_properties(dev).L2_cache_size
    peak_i8 = pk["bf16_tflops"] * 2.0
    Ms = Ms or VS_M_M
    shapes = shapes or VS_M_SHAPES
    pts = []
    gemm_only = []
    for si, (K, N) in enumerate(shapes):
        copies = min(700, max(2, -(-2 * l2 // (N * K // 4))))
        w = synth.ternary_weights(N, K, 0.35, 4100 + si)
        packed1 = vla.pack_weights(torch.from_numpy(w).to(dev))
        ring = packed1.unsqueeze(0).repeat(copies, 1).contiguous()
        del w, packed1
        beta = torch.tensor([0.05], dtype=torch.float32, device=dev)
        Mmax = max(Ms)
        xb = synth.activations(Mmax, K, 504500 + si)
        x_all = torch.from_numpy(xb.view(np.int16)).to(dev).view(torch.bfloat16)
        for M in Ms:
            x = x_all[:M].contiguous()
            out = torch.empty((M, N), dtype=torch.float32, device=dev)
            xq = torch.empty((M, K), dtype=torch.int8, device=dev)
            xs = torch.empty((M,), dtype=torch.float32, device=dev)
            ncall = copies if M <= 1024 else min(copies, 16)      # (large M: the activations alone exceed L2)

            def calls():
                for c in range(ncall):
                    vla.vla_ternary_linear(ring[c], beta, x, M, N, K, out, vla.VLA_F32, vla.VLA_PATH_AUTO, xq, xs, None, 0)
            calls()
            torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g):
                calls()
            sec = _time(torch, g.replay, 3) / ncall
            by = N * K // 4 + 4 + 2 * M * K + 4 * M * N
            op = 2.0 * M * N * K
            t_mem, t_cmp = by / (pk["hbm_gbs"] * 1e9), op / (peak_i8 * 1e12)
            p = {"M": M, "K": K, "N": N, "us": sec * 1e6, "TOPS": op / sec / 1e12, "GBs": by / sec / 1e9,
                 "roofline_frac": max(t_mem, t_cmp) / sec, "bound": "hbm" if t_mem > t_cmp else "tensor",
                 "path": int(vla.vla_ternary_auto_path(M, N, K)), "route": "single vla_ternary_linear call"}
            if p["bound"] == "tensor":
                p["frac_of_probe"] = (op / (int8_probe_tops * 1e12)) / sec
            del g
            # program route: the ring as independent stages of ONE persistent launch (M <= 16: program_kernel, IMMA;
            # M > 16: lprog_kernel, tcgen05, activation quant fused into the launch)
            nst = min(copies, 128, max(2, int(1.0e9 // (4 * M * N))))
            outs = [torch.empty((M, N), dtype=torch.float32, device=dev) for _ in range(nst)]
            stages = [dict(x=x, M=M, K=K, depends=0,
                           linears=[dict(packed=ring[c], w_scale=beta, out=outs[c], N=N, out_dtype=vla.VLA_F32)])
                      for c in range(nst)]
            prog = vla.compile_program(stages, dev)
            secp = _time(torch, lambda: vla.vla_program_run(prog), 5 if M <= 1024 else 2) / nst
            p["program_us"] = secp * 1e6
            p["program_GBs"] = by / secp / 1e9
            p["program_TOPS"] = op / secp / 1e12
            p["program_roofline_frac"] = max(t_mem, t_cmp) / secp
            p["program_stages_per_launch"] = nst
            vla.vla_program_release(prog)
            del prog, outs
            if M == synth.PREFILL_M and (K, N) in synth.MODEL_SHAPES:
                def gcalls():
                    for c in range(ncall):
                        vla.vla_ternary_gemm(ring[c], beta, xq, xs, M, N, K, out, vla.VLA_F32, vla.VLA_PATH_AUTO, None, 0)
                gcalls()
                torch.cuda.synchronize()
                gg = torch.cuda.CUDAGraph()
                with torch.cuda.graph(gg):
                    gcalls()
                gemm_only.append((op, _time(torch, gg.replay, 3) / ncall))
                del gg
            pts.append(p)
        del ring, x_all
        torch.cuda.empty_cache()
    roof_lp = None
    if synth.PREFILL_M in Ms:
        # the configs[2] prefill step (four model shapes at M = 544, Eq. 4 end to end with the quant fused) as stages of ONE
        # persistent tcgen05 launch: `nstep` steps per launch, every stage on its own cold packed-weight copy
        M, nstep = synth.PREFILL_M, 12
        rings, xs_, ops = [], [], 0.0
        for si, (K, N) in enumerate(synth.MODEL_SHAPES):
            w = synth.ternary_weights(N, K, 0.35, 4100 + si)
            packed1 = vla.pack_weights(torch.from_numpy(w).to(dev))
            rings.append(packed1.unsqueeze(0).repeat(nstep, 1).contiguous())
            xb = synth.activations(M, K, 504500 + si)
            xs_.append(torch.from_numpy(xb.view(np.int16)).to(dev).view(torch.bfloat16))
            ops += 2.0 * M * N * K
            del w, packed1
        beta = torch.tensor([0.05], dtype=torch.float32, device=dev)
        outs = [torch.empty((M, N), dtype=torch.float32, device=dev) for (K, N) in synth.MODEL_SHAPES]
        stages = [dict(x=xs_[si], M=M, K=K, depends=0,
                       linears=[dict(packed=rings[si][c], w_scale=beta, out=outs[si], N=N, out_dtype=vla.VLA_F32)])
                  for c in range(nstep)
                  for si, (K, N) in sorted(enumerate(synth.MODEL_SHAPES), key=lambda t: -t[1][0] * t[1][1])]   # largest first
        flush = torch.empty(2 * l2, dtype=torch.uint8, device=dev)
        prog = vla.compile_program(stages, dev)
        vla.vla_program_run(prog)
        torch.cuda.synchronize()
        ts = []
        for _ in range(5):
            flush.fill_(1)                                            # the packed weights leave L2 between launches
            e0, e1 = _events(torch)
            e0.record()
            vla.vla_program_run(prog)
            e1.record()
            e1.synchronize()
            ts.append(e0.elapsed_time(e1) * 1e-3)
        sec = float(np.median(ts)) / nstep
        ach = ops / sec / 1e12
        roof_lp = {"bound": "tensor", "achieved": ach, "peak": peak_i8, "unit": "TOP/s", "frac": ach / peak_i8,
                   "kernel": "lprog_kernel", "alg_ops_per_launch": ops * nstep, "us_per_launch": sec * nstep * 1e6,
                   "us_per_step": sec * 1e6,
                   "workload": "configs[2] prefill step (the four model shapes at M=544, activation quant fused, fp32 out), "
                               "%d steps = %d independent stages per persistent launch, cold weights" % (nstep, 4 * nstep),
                   "peak_source": "MEASURED_PEAKS.json bf16_tflops x 2 (int8:bf16 nominal ratio)",
                   "int8_probe_tops": int8_probe_tops, "frac_of_probe": ach / int8_probe_tops}
        vla.vla_program_release(prog)
        del prog, rings, outs, flush
        torch.cuda.empty_cache()
    roof_t = None
    if gemm_only:
        ops = sum(o for o, _ in gemm_only) / len(gemm_only)
        sec = sum(s for _, s in gemm_only) / len(gemm_only)
        ach = ops / sec / 1e12
        roof_t = {"bound": "tensor", "achieved": ach, "peak": peak_i8, "unit": "TOP/s", "frac": ach / peak_i8,
                  "kernel": "gemm_large_kernel", "alg_ops_per_launch": ops, "us_per_launch": sec * 1e6,
                  "workload": "the four model shapes at M=544, pre-quantised activations, cold weights",
                  "peak_source": "MEASURED_PEAKS.json bf16_tflops x 2 (int8:bf16 nominal ratio)",
                  "int8_probe_tops": int8_probe_tops, "frac_of_probe": ach / int8_probe_tops}
    if roof_lp is not None:
        # the product path of the prefill step is the fused persistent launch; the GEMM kernel alone stays beside it
        roof_lp["gemm_only"] = roof_t
        roof_t = roof_lp
    return pts, roof_t


# ----------------------------------------------------------------------------- cached attention
def attention_points(pk, cpu_seconds=1.0):
    """vla_cached_attention (Eq. 2) at the configs[3] head shape (20 query / 5 KV heads x 128) over a
    cached 544-token conditioning sequence, Mq in {8, 16} action queries per solver step, T steps per CUDA graph (K_C / V_C
    are computed once and stay in L2: that is the point of the cache).  Returns a list of records: us per step, the
    algorithmic bytes a step touches (Q + K_C + V_C + out) per second, GFLOP/s, and the oracle's time beside it."""
    import torch
    from paper_2606_08094_b200 import binding as vla, synth
    from oracle import attention as att
    dev = torch.device("cuda", torch.cuda.current_device())
    Hq, Hkv, d = synth.ATTN_HEADS
    Mc, T = synth.ATTN_MC, 64
    recs = []
    for Mq in (8, 16):
        q, kc, vc, _ = synth.attention_inputs(Mq, Mc, Hq, Hkv, d, 8100 + Mq)
        tb = lambda b: torch.from_numpy(np.ascontiguousarray(b).view(np.int16)).to(dev).view(torch.bfloat16)
        qd, kd, vd = tb(q), tb(kc), tb(vc)
        out = torch.empty((Mq, Hq * d), dtype=torch.bfloat16, device=dev)
        nb = vla.vla_cached_attention_workspace_bytes(Mq, Mc, Hq, Hkv, d)
        ws = torch.empty(max(nb, 16), dtype=torch.uint8, device=dev)

        def steps():
            for _ in range(T):
                vla.vla_cached_attention(qd, kd, vd, None, Mq, Mc, Hq, Hkv, d, out, vla.VLA_BF16, ws, nb)
        steps()
        torch.cuda.synchronize()
        n0 = vla.vla_launch_count()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            steps()
        launches = (vla.vla_launch_count() - n0) / T
        sec = _time(torch, g.replay, 10) / T
        by = 2 * (Mq * Hq * d + 2 * Mc * Hkv * d + Mq * Hq * d)
        fl = 4.0 * Mq * Mc * d * Hq
        t0 = time.perf_counter()
        n = 0
        while time.perf_counter() - t0 < cpu_seconds:
            att.cached_attention(q, kc, vc, Hq, Hkv, d)
            n += 1
        cpu_us = (time.perf_counter() - t0) / n * 1e6
        recs.append({"Mq": Mq, "Mc": Mc, "heads": "%dq/%dkv x %d" % (Hq, Hkv, d), "us_per_step": sec * 1e6,
                     "launches_per_step": launches, "GBs": by / sec / 1e9, "GFLOPs": fl / sec / 1e9,
                     "bound": "latency (1.4 MB of cached K_C/V_C from L2, 0.09 GFLOP)",
                     "hbm_time_us_if_uncached": by / (pk["hbm_gbs"] * 1e9) * 1e6,
                     "oracle_us_per_step": cpu_us, "oracle": "numpy float64, oracle/attention.py"})
    return recs
