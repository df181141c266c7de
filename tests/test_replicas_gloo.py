"""N > 1 path of bench.py on CPU: the path does not shard ("replicas only"), so the only multi-rank
logic is the aggregation rule -- step time = max over ranks, value = world * tokens / that time.  Two gloo ranks."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms_local = 2.0 if rank == 0 else 3.5            # the slower replica sets the job's step time
    ms, value = bench.replicas_aggregate(ms_local, 32768, dist, "cpu")
    dist.barrier()
    if rank == 0:
        out.put((ms, value))
    dist.destroy_process_group()


def test_replicas_aggregate_two_gloo_ranks():
    ctx = mp.get_context("spawn")
    out = ctx.SimpleQueue()
    port = 29500 + os.getpid() % 1000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    ms, value = out.get()
    assert ms == 3.5
    assert abs(value - 2 * 32768 / 3.5e-3) < 1e-6 * value


def test_replicas_aggregate_single_rank():
    import bench
    ms, value = bench.replicas_aggregate(1.25, 1000)
    assert ms == 1.25 and abs(value - 1000 / 1.25e-3) < 1e-9 * value
