"""Multi-GPU is "replicas only": the only cross-rank logic is bench.py's aggregation — time = MAX
over ranks, work = SUM over ranks.  Covered here with world_size 2 on the gloo backend (CPU)."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms_local = 10.0 if rank == 0 else 12.5          # rank 1 is the slow one
        ms, value = bench.aggregate(ms_local, 1_000_000, 5, dist, "cpu")
        out[rank] = (ms, value)
    finally:
        dist.destroy_process_group()


def test_aggregate_world_size_2_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Manager().dict()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    for r in range(2):
        ms, value = out[r]
        assert ms == 12.5                                # max over ranks
        assert value == pytest.approx(2 * 1_000_000 * 5 / 12.5e-3 / 1e9)   # all ranks' nodes / slowest rank's time


def test_aggregate_single_process():
    sys.path.insert(0, ROOT)
    import bench
    ms, value = bench.aggregate(4.0, 2_000_000, 10)
    assert ms == 4.0 and value == pytest.approx(2_000_000 * 10 / 4e-3 / 1e9)
