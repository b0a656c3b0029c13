"""The N > 1 path of bench.py is "replicas only" (BASELINE.json: one GPU, no sharding, no collectives):
what crosses ranks is the max of the timed region and the sum of the cells.  World size 2 over gloo, on CPU."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms, cells = bench.aggregate_replicas(10.0 + 5.0 * rank, 1000 * (rank + 1), world, torch.device("cpu"))
    dist.barrier()
    dist.destroy_process_group()
    out.put((rank, ms, cells))


def test_replica_aggregation_world2_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, 29533, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res == [(0, 15.0, 3000.0), (1, 15.0, 3000.0)]      # max of the times, sum of the cells, on every rank


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate_replicas(12.5, 7, 1, None) == (12.5, 7.0)
