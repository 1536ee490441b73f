"""N > 1 path of bench.py on CPU: two gloo ranks run the replica aggregation (max-over-ranks time,
whole-job throughput).  The path does not shard, so this
host logic is all there is to the multi-process run besides NCCL's barrier."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    local_ms = 10.0 if rank == 0 else 12.5          # rank 1 is the slow replica
    ms, mlups = bench.aggregate_over_ranks(local_ms, 1_000_000 * 20, world, "cpu")
    dist.barrier()
    out.put((rank, ms, mlups))
    dist.destroy_process_group()


def test_replica_aggregation_world_size_2():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for rank, ms, mlups in res:
        assert ms == 12.5                              # max over ranks, on every rank
        assert abs(mlups - 2 * 20.0 / 12.5e-3) < 1e-6  # both replicas' updates / slowest time
