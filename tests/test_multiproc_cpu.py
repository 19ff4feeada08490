"""N > 1 plumbing of bench.py on CPU: two processes over gloo (127.0.0.1), the barrier and the max-over-ranks /
sum-over-ranks reduction the replicas-only scaling run uses (no data-path collective)."""
import os
import socket
import sys

import torch
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    sys.path.insert(0, ROOT)
    import bench
    w, r, local = bench.dist_setup(world)
    assert (w, r, local) == (world, rank, rank)
    bench.dist_barrier(w)
    # rank r "measured" (10 + r) ms and processed (100 * (r + 1)) units
    t, u = bench.reduce_max_and_sum(w, 10.0 + r, 100.0 * (r + 1), torch.device("cpu"))
    bench.dist_barrier(w)
    out.put((rank, t, u))
    import torch.distributed as dist
    dist.destroy_process_group()


def test_two_rank_gloo_max_time_sum_units():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, t, u in res:
        assert t == 11.0          # max over ranks of the time
        assert u == 300.0         # whole-job units = sum over ranks


def test_reference_arm_runs_on_rank0_only(monkeypatch):
    """--impl reference under torchrun: every rank but 0 exits 0 without work."""
    sys.path.insert(0, ROOT)
    import bench
    monkeypatch.setenv("RANK", "1")

    class A:
        workload, gpus, steps, warmup = "decode", 2, 1, 0
    assert bench.run_reference(A()) == 0
