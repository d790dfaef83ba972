"""N > 1 path of bench.py ("replicas only", no data-path collective): the only cross-rank step is the timing
reduction (max seconds over ranks, sum of units).  Covered here with world_size 2 over gloo on CPU."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    assert bench.rank_info() == (rank, rank, world)
    secs, units = bench.reduce_over_ranks(1.0 + rank, 100.0 * (rank + 1), world, dist)
    q.put((rank, secs, units))
    dist.barrier()
    dist.destroy_process_group()


def test_reduce_over_ranks_world2_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, secs, units in res:
        assert secs == 2.0 and units == 300.0      # max over ranks of the time, sum of the units


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks(1.5, 10.0, 1) == (1.5, 10.0)
    assert abs(bench.PEAK_TFLOPS_DERIVED - 37.2) < 0.1
