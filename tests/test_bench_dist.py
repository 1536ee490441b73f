"""N > 1 host logic of bench.py on CPU: two gloo ranks run the aggregation both multi-rank modes use
(max-over-ranks time, whole-job throughput).  The sharded step itself (bench.py's default for
N > 1: z-slabs) is covered by tests/test_slab_host.py (halo lists, ring
choreography on two gloo ranks) and tests/test_gpu_slab.py; here also the mode selection."""
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


def test_mode_selection(monkeypatch):
    """One GPU: the headline workload (config 4), plain step.  torchrun with N > 1: the sharded
    path on config 5, unless --shard replicas / --config say otherwise."""
    sys.path.insert(0, ROOT)
    import bench
    monkeypatch.setattr(sys, "argv", ["bench.py"])
    a = bench.parse_args()
    assert a.shard is None and a.config is None and a.gpus == 1
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "8", "--shard", "replicas", "--config", "4"])
    a = bench.parse_args()
    assert (a.shard, a.config, a.gpus) == ("replicas", 4, 8)
    src = open(os.path.join(ROOT, "bench.py")).read()
    assert 'shard = a.shard or ("slab" if world > 1 else "replicas")' in src


def test_roofline_traffic_is_keyed_by_the_build():
    """bench.py reports roofline.traffic only from an ncu capture of the build it runs
    (profiles/ncu_traffic.csv keyed by the source hash), never a number of another build."""
    sys.path.insert(0, ROOT)
    import bench
    sha = bench.source_sha16()
    assert len(sha) == 16
    rows = [l for l in open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")) if not l.startswith("#")]
    assert rows and all(len(l.split(", ")) == 4 for l in rows)
    k = "k_collide_stream_bulk<float,128,7,1,1>"
    got = bench.ncu_traffic("cfg4_grf_256_imbibition", k)
    mine = [l for l in rows if l.startswith(sha)]
    if mine:
        assert got is not None and 1.3e9 < got < 1.7e9      # 312 B x N_f = 1.352 GB + index
    else:
        assert got is None
    assert bench.ncu_traffic("cfg5_spherepack_512_throughput", k) is None
    assert bench.ncu_traffic(None, k) is None
