"""The N > 1 path of bench.py is "replicas only" (Multi-GPU): every rank steps its own copy and the
only exchange is the max-over-ranks of the timing.  Covered here with two gloo processes on the CPU."""
import os
import sys

import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    local_ms = 10.0 if rank == 0 else 25.0  # the slower replica decides
    value, ms = bench.whole_job_value(points=1000, steps=4, ms_local=local_ms, world=world)
    out[rank] = (value, ms)
    dist.destroy_process_group()


def test_whole_job_value_is_max_over_ranks():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, 29591, out), nprocs=world, join=True)
        res = dict(out)
    for r in range(world):
        value, ms = res[r]
        assert ms == 25.0
        assert abs(value - world * 1000 * 4 / 25e-3) < 1e-6


def test_single_rank_needs_no_group():
    sys.path.insert(0, ROOT)
    import bench
    value, ms = bench.whole_job_value(points=10, steps=2, ms_local=4.0, world=1)
    assert ms == 4.0 and abs(value - 10 * 2 / 4e-3) < 1e-9
