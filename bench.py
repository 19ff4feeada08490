#!/usr/bin/env python
"""bench.py -- throughput of the ternary-linear hot path (arxiv/paper_2606_08094 Eq. 4) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload decode|prefill] [--impl reference]

Workload (BASELINE.json configs[1], the default): the four BitNet-2B-class linears
(K,N) in {(2560,2560),(2560,640),(2560,6912),(6912,2560)} at M in {1,8,16}; a STEP is one pass of the
whole hot path (activation quant -> packed-weight decode -> int8 contraction -> dequant epilogue, bf16
output) over all 12 points, executed as ONE persistent launch (vla_program_run: 12 independent stages).  `--workload prefill` is configs[2] (M=544, fp32
out).  The metric is BASELINE.json's: algorithmic HBM GB/s (packed weights + bf16 activations in + outputs
out) with the TOPS (2MNK) beside it and the roofline fraction of the
dominant kernel.  Weights are kept COLD: every step reads its packed weights from the next slot of a ring
of copies whose total size exceeds twice the L2, so the GB/s are HBM GB/s, not L2 GB/s.

Timing: the launches of a step are captured in CUDA graphs (the paper's own remedy for dispatch overhead,
PAPER.md line 56) and replayed; CUDA events on the launching stream; barrier + synchronize on both sides;
max over ranks.  Multi-GPU: the path runs on one GPU (BASELINE.json north_star) -> replicas only, weak
scaling, no collective.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "ternary GEMM TOPS & HBM GB/s vs M; fraction of INT8/HBM roofline (1 B200)"      # BASELINE.json:metric
FALLBACK_HBM_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback
NOMINAL_HBM_GBS = 8000.0           # BASELINE.json north_star "~8 TB/s"
NOMINAL_INT8_TOPS = 4500.0         # dense int8, datasheet (same rate as fp8)
E2E_BUFFER_SETS = 4                # end-to-end leg: steps in flight (device + pinned host arenas and a stream each)


# ----------------------------------------------------------------------------- workload description
def workload_points(name):
    """[(M, shape_idx)] of one step, in execution order."""
    from paper_2606_08094_b200 import synth
    if name == "decode":
        return [(M, si) for M in synth.DECODE_M for si in range(len(synth.MODEL_SHAPES))]
    if name == "prefill":
        # the four independent linears, largest first: in the one-launch program the long tiles then start first and the
        # short stages fill the CTAs they leave idle (38.8 -> 34.5 us per one-step launch)
        order = sorted(range(len(synth.MODEL_SHAPES)), key=lambda si: -synth.MODEL_SHAPES[si][0] * synth.MODEL_SHAPES[si][1])
        return [(synth.PREFILL_M, si) for si in order]
    raise ValueError(name)


def workload_name(workload):
    """`config.workload` of the JSON line -- the same string for the B200 arm and the reference arm."""
    if workload == "decode":
        return "configs[1] decode: 4 BitNet-2B linears x M in {1,8,16}, fused quant, bf16 out (B200 arm: one persistent program launch per step)"
    return "configs[2] prefill: 4 BitNet-2B linears at M=544, fused quant, fp32 out (B200 arm: one persistent tcgen05 program launch per step)"


def out_elem_bytes(workload):
    return 2 if workload == "decode" else 4       # configs[1]: bf16 output; configs[2]: fp32 output


def point_bytes(M, K, N, out_bytes, fused_quant=True):
    """Algorithmic bytes of one call: packed W + beta + X in + Y out."""
    x_in = 2 * M * K if fused_quant else M * K + 4 * M
    return N * K // 4 + 4 + x_in + M * N * out_bytes


def point_ops(M, K, N):
    return 2 * M * N * K


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), bf16_tflops=float(d.get("bf16_tflops", 0.0)),
                    bf16_tflops_sustained=float(d.get("bf16_tflops_sustained", 0.0)), source="measured")
    return dict(hbm_gbs=FALLBACK_HBM_GBS, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, source="fallback")


def ncu_traffic(kernel_key):
    """DRAM bytes per launch of the dominant kernel from the committed ncu capture, or None."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")      # kernel,dram_bytes_per_launch,capture
    if os.path.exists(p):
        for line in open(p).read().splitlines()[1:]:
            f = line.split(",")
            if len(f) >= 2 and f[0] == kernel_key:
                return float(f[1])
    return None


# ----------------------------------------------------------------------------- clocks sampler
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "50"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [t.strip() for t in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["no samples"])
        return dict(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons),
                    samples=len(sm))


# ----------------------------------------------------------------------------- reference arm (the oracle)
def oracle_step_inputs(workload):
    from paper_2606_08094_b200 import synth
    pts = []
    cache = {}
    for (M, si) in workload_points(workload):
        c = synth.config1_point(si, M) if workload == "decode" else synth.config2_point(si)
        if si in cache:
            c["w"] = cache[si]
        cache[si] = c["w"]
        pts.append(c)
    return pts


def oracle_time_steps(workload, pts, steps, budget_s=None, row_cap=None):
    """Times the oracle, as it stands, on `steps` passes over the points (optionally only the first row_cap
    rows of each point's activations: a bounded sample).  Returns (seconds, steps_done, bytes, ops)."""
    from oracle import oracle as orc
    ob = out_elem_bytes(workload)
    nbytes = nops = 0
    t0 = time.perf_counter()
    done = 0
    for _ in range(steps):
        for c in pts:
            x = c["x"] if row_cap is None else c["x"][:row_cap]
            M = x.shape[0]
            orc.ternary_linear(x, c["w"], c["beta"], want_y64=False)
            nbytes += point_bytes(M, c["K"], c["N"], ob)
            nops += point_ops(M, c["K"], c["N"])
        done += 1
        if budget_s is not None and time.perf_counter() - t0 > budget_s:
            break
    return time.perf_counter() - t0, done, nbytes, nops


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import oracle as orc
    orc.build()
    pts = oracle_step_inputs(args.workload)
    cap = None if args.workload == "decode" else 32      # prefill: 32 of the 544 rows per point per step
    oracle_time_steps(args.workload, pts, min(args.warmup, 1), row_cap=cap)
    sec, done, nbytes, nops = oracle_time_steps(args.workload, pts, args.steps, budget_s=150.0, row_cap=cap)
    val = nbytes / sec / 1e9
    sample = "all 12 points, all rows" if cap is None else "first %d rows of each of the 4 points" % cap
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": "GB/s",
        "n_gpus": args.gpus, "steps": done, "warmup": min(args.warmup, 1), "ms_per_step": sec / done * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int8*ternary->int32",
        "data": "synthetic", "tops": nops / sec / 1e12,
        "config": {"workload": workload_name(args.workload), "sample": sample},
        "cpu_baseline": {"value": val, "unit": "GB/s", "cores": orc.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------- distributed plumbing
def dist_setup(n_gpus):
    import torch
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        backend = "nccl" if torch.cuda.is_available() else "gloo"
        dist.init_process_group(backend=backend)
    return world, rank, local


def dist_barrier(world):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def reduce_max_and_sum(world, t_local, units_local, device):
    """max over ranks of the time, sum over ranks of the units (replicas: whole-job units / slowest rank)."""
    import torch
    if world == 1:
        return t_local, units_local
    import torch.distributed as dist
    t = torch.tensor([t_local], dtype=torch.float64, device=device)
    u = torch.tensor([units_local], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


# ----------------------------------------------------------------------------- GPU arm
class GpuWorkload:
    """Device-resident state of one workload: a ring of packed-weight copies per shape (cold weights), and per
    point the activation / output / workspace buffers plus pinned host mirrors for the end-to-end leg."""

    def __init__(self, vla, workload, device):
        import torch
        from paper_2606_08094_b200 import synth
        self.vla, self.torch, self.workload, self.device = vla, torch, workload, device
        self.points = workload_points(workload)
        self.out_dtype = vla.VLA_BF16 if workload == "decode" else vla.VLA_F32
        self.out_bytes = out_elem_bytes(workload)
        self.uses = max(1, len(self.points) // len(synth.MODEL_SHAPES))       # times a shape is used per step
        l2 = torch.cuda.get_device_properties(device).L2_cache_size
        per_copy = sum(n * k // 4 for (k, n) in synth.MODEL_SHAPES)
        copies = -(-2 * l2 // per_copy)
        copies = -(-copies // self.uses) * self.uses
        self.copies, self.rev_steps, self.l2 = copies, copies // self.uses, l2
        self.ring, self.beta = [], []
        xs_full = {}
        for si, (K, N) in enumerate(synth.MODEL_SHAPES):
            c = synth.config1_point(si, max(synth.DECODE_M)) if workload == "decode" else synth.config2_point(si)
            w = torch.from_numpy(c["w"]).to(device)
            packed = vla.pack_weights(w)
            self.ring.append(packed.unsqueeze(0).repeat(copies, 1).contiguous())
            self.beta.append(torch.tensor([float(c["beta"])], dtype=torch.float32, device=device))
            xs_full[si] = c["x"]
            del w
        self.buf = []
        # All activation inputs of a step live in ONE device arena (and one pinned host arena), all outputs in another:
        # the host-buffer call then moves a step's inputs with one copy and its outputs with one copy.
        dt = torch.bfloat16 if self.out_dtype == vla.VLA_BF16 else torch.float32
        esz = 2 if dt == torch.bfloat16 else 4
        al = lambda n: -(-n // 256) * 256
        x_off, o_off, xo, oo = [], [], 0, 0
        for (M, si) in self.points:
            K, N = synth.MODEL_SHAPES[si]
            x_off.append(xo); xo += al(2 * M * K)
            o_off.append(oo); oo += al(esz * M * N)
        self.x_arena = torch.empty(xo, dtype=torch.uint8, device=device)
        self.x_arena_host = torch.empty(xo, dtype=torch.uint8).pin_memory()
        self.o_arena = torch.empty(oo, dtype=torch.uint8, device=device)
        self.o_arena_host = torch.empty(oo, dtype=torch.uint8).pin_memory()
        for pi, (M, si) in enumerate(self.points):
            K, N = synth.MODEL_SHAPES[si]
            xb = np.ascontiguousarray(xs_full[si][:M])
            x_host = self.x_arena_host[x_off[pi]:x_off[pi] + 2 * M * K].view(torch.bfloat16).view(M, K)
            x_host.copy_(torch.from_numpy(xb.view(np.int16)).view(torch.bfloat16))
            x_dev = self.x_arena[x_off[pi]:x_off[pi] + 2 * M * K].view(torch.bfloat16).view(M, K)
            x_dev.copy_(x_host)
            out_dev = self.o_arena[o_off[pi]:o_off[pi] + esz * M * N].view(dt).view(M, N)
            out_host = self.o_arena_host[o_off[pi]:o_off[pi] + esz * M * N].view(dt).view(M, N)
            ws_bytes = vla.vla_ternary_host_workspace_bytes(M, N, K, self.out_dtype)
            self.buf.append(dict(
                M=M, K=K, N=N, si=si, x=x_dev, x_host=x_host,
                out=out_dev, out_host=out_host,
                xq=torch.empty((M, K), dtype=torch.int8, device=device),
                xs=torch.empty((M,), dtype=torch.float32, device=device),
                ws=torch.empty(ws_bytes, dtype=torch.uint8, device=device), ws_bytes=ws_bytes))
        # the points of a step are one compiled program per ring position: ONE persistent launch per step
        # (decode: program_kernel, M <= 16; prefill: lprog_kernel, tcgen05, activation quant fused into the launch)
        self.programs = []
        if workload in ("decode", "prefill"):
            for step in range(self.rev_steps):
                stages = [dict(x=b["x"], M=b["M"], K=b["K"], depends=0,
                               linears=[dict(packed=self.ring[b["si"]][self.slot(step, pi)], w_scale=self.beta[b["si"]],
                                             out=b["out"], N=b["N"], out_dtype=self.out_dtype)])
                          for pi, b in enumerate(self.buf)]
                self.programs.append(vla.compile_program(stages, device))
            self.copies_in = vla.make_copies([(self.x_arena_host, self.x_arena)])
            self.copies_out = vla.make_copies([(self.o_arena_host, self.o_arena)])
        self.step_bytes = sum(point_bytes(b["M"], b["K"], b["N"], self.out_bytes) for b in self.buf)
        self.step_ops = sum(point_ops(b["M"], b["K"], b["N"]) for b in self.buf)
        self.gemm_bytes = sum(point_bytes(b["M"], b["K"], b["N"], self.out_bytes, fused_quant=False) for b in self.buf)
        self.h2d = sum(2 * b["M"] * b["K"] for b in self.buf)
        self.d2h = sum(self.out_bytes * b["M"] * b["N"] for b in self.buf)

    def build_pipeline(self, nbuf=2):
        """End-to-end serving loop: `nbuf` buffer sets (device arenas, pinned host arenas, programs on those arenas), one
        stream each, so that the copies of neighbouring steps overlap the kernel (vla_program_run_host_async)."""
        torch, vla = self.torch, self.vla
        self.pipe = []
        for b in range(nbuf):
            x_dev = torch.empty_like(self.x_arena)
            o_dev = torch.empty_like(self.o_arena)
            x_host = torch.empty(self.x_arena_host.numel(), dtype=torch.uint8).pin_memory()
            o_host = torch.empty(self.o_arena_host.numel(), dtype=torch.uint8).pin_memory()
            x_host.copy_(self.x_arena_host)
            progs = []
            for step in range(self.rev_steps):
                stages = []
                for pi, bf in enumerate(self.buf):
                    xo = bf["x"].data_ptr() - self.x_arena.data_ptr()
                    oo = bf["out"].data_ptr() - self.o_arena.data_ptr()
                    xv = x_dev[xo:xo + bf["x"].numel() * 2].view(torch.bfloat16).view(bf["M"], bf["K"])
                    ov = o_dev[oo:oo + bf["out"].numel() * bf["out"].element_size()].view(bf["out"].dtype).view(bf["M"], bf["N"])
                    stages.append(dict(x=xv, M=bf["M"], K=bf["K"], depends=0,
                                       linears=[dict(packed=self.ring[bf["si"]][self.slot(step, pi)], w_scale=self.beta[bf["si"]],
                                                     out=ov, N=bf["N"], out_dtype=self.out_dtype)]))
                progs.append(vla.compile_program(stages, x_dev.device))
            self.pipe.append(dict(x_dev=x_dev, o_dev=o_dev, x_host=x_host, o_host=o_host, progs=progs,
                                  cin=vla.make_copies([(x_host, x_dev)]), cout=vla.make_copies([(o_host, o_dev)]),
                                  stream=torch.cuda.Stream()))

    def run_pipeline(self, steps):
        """`steps` end-to-end steps, round robin over the buffer sets; a set is reused only after its previous step's
        results have arrived on the host (event synchronise: that is where a server would read them and write new inputs)."""
        vla = self.vla
        call, ok = vla._lib.vla_program_run_host_async, vla.VLA_OK
        nb, rev = len(self.pipe), self.rev_steps
        for p in self.pipe:                                   # marshal once: raw pointers, one reusable event per set
            if "ptrs" not in p:
                p["ptrs"] = [int(g.data_ptr()) for g in p["progs"]]
                p["sptr"] = p["stream"].cuda_stream
                p["ev"] = self.torch.cuda.Event()
                p["busy"] = False
        for s in range(steps):
            p = self.pipe[s % nb]
            if p["busy"]:
                p["ev"].synchronize()
            st = call(p["ptrs"][s % rev], p["cin"], 1, p["cout"], 1, p["sptr"])
            if st != ok:
                raise vla.VlaError(st, "vla_program_run_host_async")
            p["ev"].record(p["stream"])
            p["busy"] = True
        for p in self.pipe:
            if p["busy"]:
                p["ev"].synchronize()
                p["busy"] = False

    def slot(self, step, pi):
        return (step * self.uses + pi // 4) % self.copies

    def launch_point(self, pi, step, mode="linear"):
        b, vla = self.buf[pi], self.vla
        packed = self.ring[b["si"]][self.slot(step, pi)]
        if mode in ("linear", "calls"):   # the whole hot path as single calls: quant kernel + GEMM kernel per linear
            vla.vla_ternary_linear(packed, self.beta[b["si"]], b["x"], b["M"], b["N"], b["K"], b["out"], self.out_dtype,
                                   vla.VLA_PATH_AUTO, b["xq"], b["xs"], b["ws"], b["ws_bytes"])
        elif mode == "gemm":          # the dominant kernel alone, on pre-quantised activations
            vla.vla_ternary_gemm(packed, self.beta[b["si"]], b["xq"], b["xs"], b["M"], b["N"], b["K"], b["out"],
                                 self.out_dtype, vla.VLA_PATH_AUTO, b["ws"], b["ws_bytes"])
        elif mode == "host":          # end to end: pinned host x -> device -> kernels -> pinned host y, synchronised
            vla.vla_ternary_linear_host(packed, self.beta[b["si"]], b["x_host"], b["M"], b["N"], b["K"], b["out_host"],
                                        self.out_dtype, vla.VLA_PATH_AUTO, b["ws"], b["ws_bytes"])

    def launch_step(self, step, mode="linear", only=None):
        if self.programs and only is None and mode in ("linear", "host"):
            prog = self.programs[step % self.rev_steps]
            if mode == "linear":
                self.vla.vla_program_run(prog)
            else:
                self.vla.vla_program_run_host(prog, self.copies_in, self.copies_out)
            return
        for pi in range(len(self.buf)):
            if only is None or pi == only:
                self.launch_point(pi, step, mode)

    def capture(self, steps, mode="linear", only=None):
        """CUDA graph of `steps` = [step indices]; returns (graph, kernels launched per replay)."""
        torch = self.torch
        n0 = self.vla.vla_launch_count()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            for s in steps:
                self.launch_step(s, mode, only)
        return g, self.vla.vla_launch_count() - n0


def time_replays(torch, plan):
    """plan: list of graphs to replay in order.  Returns milliseconds (CUDA events on the current stream)."""
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for g in plan:
        g.replay()
    e1.record()
    e1.synchronize()
    return e0.elapsed_time(e1)


def run_gpu(args):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU path (use --impl reference for the oracle)")
    from paper_2606_08094_b200 import binding as vla
    world, rank, local = dist_setup(args.gpus)
    device = torch.device("cuda", local)
    torch.cuda.set_device(device)
    wl = GpuWorkload(vla, args.workload, device)
    rev = wl.rev_steps

    # warm-up, eager (also sets function attributes outside any capture)
    for s in range(max(args.warmup, 3)):
        wl.launch_step(s)
        if args.workload != "decode":
            wl.launch_step(s, "calls")
            wl.launch_step(s, "gemm")
    torch.cuda.synchronize()

    g_rev, n_rev = wl.capture(list(range(rev)))
    singles = {}
    plan, launches = [], 0
    full, rem = divmod(args.steps, rev)
    plan += [g_rev] * full
    launches += n_rev * full
    for s in range(rem):
        singles[s], n1 = wl.capture([s])
        plan.append(singles[s])
        launches += n1
    warm_plan = [g_rev] * max(1, -(-args.warmup // rev))
    time_replays(torch, warm_plan)

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.12)
    torch.cuda.synchronize()
    dist_barrier(world)
    ms_local = time_replays(torch, plan)
    torch.cuda.synchronize()
    dist_barrier(world)
    clocks = sampler.stop() if rank == 0 else None
    ms, total_bytes = reduce_max_and_sum(world, ms_local, float(wl.step_bytes) * args.steps, device)
    _, total_ops = reduce_max_and_sum(world, ms_local, float(wl.step_ops) * args.steps, device)

    # ---- end-to-end leg: host buffers through the C ABI, copies inside the timed region
    e2e_steps = max(3, min(args.steps, args.e2e_steps))
    for s in range(3):
        wl.launch_step(s, "host")
    torch.cuda.synchronize()
    dist_barrier(world)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for s in range(e2e_steps):
        wl.launch_step(s, "host")
    e1.record()
    e1.synchronize()
    dist_barrier(world)
    e2e_sync_ms, _ = reduce_max_and_sum(world, e0.elapsed_time(e1), float(wl.step_bytes) * e2e_steps, device)
    # the same, pipelined: two buffer sets on two streams (vla_program_run_host_async), host wall clock around the loop
    wl.build_pipeline(E2E_BUFFER_SETS)
    wl.run_pipeline(4)
    torch.cuda.synchronize()
    dist_barrier(world)
    t0 = time.perf_counter()
    wl.run_pipeline(e2e_steps)
    torch.cuda.synchronize()
    pipe_ms = (time.perf_counter() - t0) * 1e3
    dist_barrier(world)
    e2e_ms, e2e_bytes = reduce_max_and_sum(world, pipe_ms, float(wl.step_bytes) * e2e_steps, device)
    for p in wl.pipe:                                         # the pipelined leg computed the same step: check its results
        for bf in wl.buf:
            oo = bf["out"].data_ptr() - wl.o_arena.data_ptr()
            nb = bf["out"].numel() * bf["out"].element_size()
            assert torch.equal(p["o_host"][oo:oo + nb], bf["out_host"].view(-1).view(torch.uint8)), \
                "pipelined end-to-end output differs from the synchronous call's"

    if rank != 0:
        return 0

    # ---- roofline of the dominant kernel (the GEMM), timed alone on pre-quantised activations, cold ring
    pk = peaks()
    # the dominant (only) kernel of the step is the persistent program kernel: one launch = one step
    g_one, n_one = wl.capture(list(range(rev)))
    time_replays(torch, [g_one] * 2)
    reps = max(3, min(200, int(4000 / max(1, rev))))
    per_launch_s = time_replays(torch, [g_one] * reps) * 1e-3 / (reps * n_one)
    if args.workload == "decode":
        alg = float(wl.step_bytes)                            # algorithmic bytes of one launch
        achieved = alg / per_launch_s / 1e9
        roof = {"bound": "hbm", "achieved": achieved, "peak": pk["hbm_gbs"], "unit": "GB/s",
                "frac": achieved / pk["hbm_gbs"], "traffic": ncu_traffic("program_kernel"),
                "kernel": "program_kernel", "peak_source": pk["source"] + " (MEASURED_PEAKS.json hbm_gbs)",
                "alg_bytes_per_launch": alg, "us_per_launch": per_launch_s * 1e6,
                "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS}
    else:
        alg = float(wl.step_ops)                              # one launch = the four linears of the step, Eq. 4 end to end
        achieved = alg / per_launch_s / 1e12
        peak_i8 = pk["bf16_tflops"] * 2.0                     # int8 : bf16 = 4.5 : 2.25 nominal
        probe = int8_probe_tops(vla)                          # tcgen05.mma.kind::i8 issue-rate ceiling of this box
        roof = {"bound": "tensor", "achieved": achieved, "peak": peak_i8, "unit": "TOP/s",
                "frac": achieved / peak_i8, "traffic": ncu_traffic("lprog_kernel"),
                "kernel": "lprog_kernel", "peak_source": pk["source"] + " bf16_tflops x 2 (int8:bf16 nominal ratio)",
                "alg_ops_per_launch": alg, "us_per_launch": per_launch_s * 1e6,
                "frac_of_nominal_4500": achieved / NOMINAL_INT8_TOPS, "int8_probe_tops": probe,
                "frac_of_probe": achieved / probe}
        # beside it: the same step as single calls (quant kernel + GEMM kernel per linear, CUDA graph + PDL), and the GEMM
        # kernel alone on pre-quantised activations
        g_calls, n_calls = wl.capture(list(range(rev)), "calls")
        time_replays(torch, [g_calls] * 2)
        calls_s = time_replays(torch, [g_calls] * 20) * 1e-3 / (20 * rev)
        g_gemm, n_gemm = wl.capture(list(range(rev)), "gemm")
        time_replays(torch, [g_gemm] * 2)
        gemm_s = time_replays(torch, [g_gemm] * 20) * 1e-3 / (20 * n_gemm)
        a_g = wl.step_ops / len(wl.buf) / gemm_s / 1e12
        roof["single_calls"] = {"us_per_step": calls_s * 1e6, "launches_per_step": n_calls // rev,
                                "TOPS": wl.step_ops / calls_s / 1e12, "frac": wl.step_ops / calls_s / 1e12 / peak_i8}
        roof["gemm_only"] = {"kernel": "gemm_large_kernel", "us_per_launch": gemm_s * 1e6, "achieved": a_g,
                             "frac": a_g / peak_i8, "frac_of_probe": a_g / probe, "traffic": ncu_traffic("gemm_large")}

    # ---- per-point table (the metric is "vs M"): each point alone, whole hot path, cold ring
    table = []
    if not args.no_points:
        for pi, b in enumerate(wl.buf):
            g, n = wl.capture(list(range(rev)), "linear", only=pi)
            time_replays(torch, [g])
            r = max(3, min(50, int(5e4 / rev)))
            t = time_replays(torch, [g] * r) * 1e-3 / (r * rev)
            by, op = point_bytes(b["M"], b["K"], b["N"], wl.out_bytes), point_ops(b["M"], b["K"], b["N"])
            t_roof = max(by / (pk["hbm_gbs"] * 1e9), op / (pk["bf16_tflops"] * 2e12))
            table.append({"M": b["M"], "K": b["K"], "N": b["N"], "us": t * 1e6, "GBs": by / t / 1e9,
                          "TOPS": op / t / 1e12, "roofline_frac": t_roof / t,
                          "path": int(vla.vla_ternary_auto_path(b["M"], b["N"], b["K"])),
                          "route": "single vla_ternary_linear call (quant kernel + GEMM kernel)"})
            del g

    # ---- the metric is "vs M": both halves (HBM-bound M <= 16, tensor-bound M >= 512) in the same line
    vs_m, roof_tensor = None, None
    if args.workload == "decode" and not args.no_vs_m:
        import bench_workloads as bw
        vs_m, roof_tensor = bw.run_vs_m(pk, int8_probe_tops(vla))
        if roof_tensor is not None:
            t1 = ncu_traffic("lprog_kernel")                # DRAM bytes of the captured ONE-step launch (--workload prefill)
            nstep = max(1, int(round(roof_tensor["us_per_launch"] / roof_tensor["us_per_step"])))
            roof_tensor["traffic"] = None if t1 is None else t1 * nstep
            roof_tensor["traffic_source"] = "DRAM bytes per step of the captured one-step launch x %d steps per launch" % nstep
            if roof_tensor.get("gemm_only"):
                roof_tensor["gemm_only"]["traffic"] = ncu_traffic("gemm_large")

    attn = None
    if args.workload == "decode" and not args.no_vs_m:
        import bench_workloads as bw
        attn = bw.attention_points(pk)                        # SURVEY 8(f) NEXT-4, reported beside the hot path

    # ---- the oracle on this box's host cores, bounded sample
    from oracle import oracle as orc
    orc.build()
    pts = oracle_step_inputs(args.workload)
    cap = None if args.workload == "decode" else 32
    oracle_time_steps(args.workload, pts, 1, row_cap=cap)
    sec, done, nbytes, nops = oracle_time_steps(args.workload, pts, 10 ** 6, budget_s=args.cpu_budget, row_cap=cap)
    cpu = {"value": nbytes / sec / 1e9, "unit": "GB/s", "cores": orc.num_threads(), "kind": "oracle",
           "sample": ("%d full steps (all 12 points, all rows)" % done) if cap is None
           else ("%d steps of the first %d rows of each of the 4 points" % (done, cap)),
           "tops": nops / sec / 1e12, "seconds": sec}

    value = total_bytes / (ms * 1e-3) / 1e9
    line = {
        "metric": METRIC, "value": value, "unit": "GB/s", "n_gpus": world,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "int8*ternary->int32", "data": "synthetic",
        "tops": total_ops / (ms * 1e-3) / 1e12,
        "config": {"workload": workload_name(args.workload),
                   "cold_weights": "ring of %d packed copies per shape (%.0f MB > 2 x L2 %.0f MB), next slot every use"
                   % (wl.copies, wl.copies * sum(r.shape[1] for r in wl.ring) / 1e6, wl.l2 / 1e6),
                   "value_is": ("algorithmic HBM GB/s of the configs[1] decode step (the M <= 16 half of the metric); both halves "
                                "per (shape, M) are in vs_M, the dominant kernel of the M >= 512 half in roofline_tensor")
                   if args.workload == "decode" else "algorithmic HBM GB/s of the configs[2] prefill step; TOPS beside it",
                   "launch": "CUDA graphs of %d program launches" % rev, "parallelism": "replicas" if world > 1 else "single"},
        "clocks": clocks, "gpu_launches": launches,
        "e2e": {"value": e2e_bytes / (e2e_ms * 1e-3) / 1e9, "unit": "GB/s", "h2d_bytes_per_step": wl.h2d,
                "d2h_bytes_per_step": wl.d2h, "steps": e2e_steps, "ms_per_step": e2e_ms / e2e_steps,
                "mode": "vla_program_run_host_async, %d buffer sets on %d streams (copies of neighbouring steps overlap the "
                        "kernel); host wall clock over the loop" % (E2E_BUFFER_SETS, E2E_BUFFER_SETS),
                "synchronous_ms_per_step": e2e_sync_ms / e2e_steps,
                "synchronous_value": float(wl.step_bytes) * world / (e2e_sync_ms / e2e_steps * 1e-3) / 1e9},
        "roofline": roof, "roofline_tensor": roof_tensor, "cpu_baseline": cpu, "points": table, "vs_M": vs_m, "attention_next4": attn,
        "step_roofline_frac_hbm": value / pk["hbm_gbs"],
    }
    print(json.dumps(line))
    return 0


def int8_probe_tops(vla):
    """Box-measured INT8 tensor ceiling: back-to-back tcgen05.mma.kind::i8 (128x256x32) on every SM, no loads."""
    import torch
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    n = 20000
    ms = vla.vla_i8_mma_issue_probe(sms, n)
    return 2.0 * 128 * 256 * 32 * n * sms / (ms * 1e-3) / 1e12


def run_extra(args):
    """configs[3] / configs[4] (single GPU; BASELINE.json north_star: everything runs on one GPU)."""
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU path (use --impl reference for the oracle)")
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    torch.cuda.set_device(0)
    from paper_2606_08094_b200 import binding as vla
    import bench_workloads as bw
    pk = peaks()
    if args.workload == "stack":
        return bw.run_stack(args, pk, ClockSampler(0))
    if args.workload == "dispatch":
        return bw.run_dispatch(args, pk, ClockSampler(0))
    return bw.run_sweep(args, pk, ClockSampler(0), int8_probe_tops(vla))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=4000)
    ap.add_argument("--warmup", type=int, default=16)
    ap.add_argument("--workload", choices=["decode", "prefill", "stack", "sweep", "dispatch"], default="decode")
    ap.add_argument("--quick", action="store_true", help="sweep: one zero fraction and one distribution only")
    ap.add_argument("--sweep-m", default="", help="sweep: comma-separated M values (default: 1,2,4,...,4096)")
    ap.add_argument("--impl", choices=["b200", "reference"], default="b200")
    ap.add_argument("--e2e-steps", type=int, default=200)
    ap.add_argument("--cpu-budget", type=float, default=12.0, help="seconds of oracle timing for cpu_baseline")
    ap.add_argument("--no-points", action="store_true", help="skip the per-point table")
    ap.add_argument("--no-vs-m", action="store_true", help="skip the vs-M block (both halves of the metric)")
    args = ap.parse_args()
    if args.impl == "reference":
        if args.workload in ("stack", "sweep", "dispatch"):
            args.workload = "decode"
        return run_reference(args)
    if args.workload in ("stack", "sweep", "dispatch"):
        return run_extra(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
