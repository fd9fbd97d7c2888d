"""world_size-2 gloo test (CPU) of bench.py's multi-rank logic: the path does not shard ("replicas only"), so the
only cross-rank step is the max-over-ranks of the device timings and the whole-job aggregation."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(100.0 + 50.0 * rank, world)        # rank 1 is the slow one
    dist.barrier()
    q.put((rank, ms, bench.aggregate(ms * 1e-3 / 4, world)))
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, agg in res:
        assert ms == 150.0                      # every rank reports the max
        assert abs(agg - 0.150 / 4 / 2) < 1e-15  # 2 replicas x 4 rhs in 150 ms


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(12.5, 1) == 12.5 and bench.aggregate(3.0, 1) == 3.0
