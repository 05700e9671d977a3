"""N > 1 path of bench.py on CPU: replicas only, so the only cross-rank logic is the
max-over-ranks of the elapsed time and the whole-job aggregate.  world_size 2, gloo backend."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, "cpu")     # rank 1 is the slow one
    out[rank] = (ms, bench.whole_job_value(world, 1000, 3, ms))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_world2():
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, 29731, out), nprocs=2, join=True)
        res = dict(out)
    assert res[0] == res[1]
    ms, value = res[0]
    assert ms == 15.0
    assert abs(value - 2 * 1000 * 3 / 15e-3 / 1e6) < 1e-12


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, None, "cpu") == 3.5
    assert bench.whole_job_value(1, 2_000_000, 3, 1.0) == 6000.0
