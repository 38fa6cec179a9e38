"""bench.py's N > 1 logic on CPU: two gloo ranks (replicas only: DESIGN.md "Multi-GPU"), time = MAX over ranks,
value = whole-job aggregate.  No GPU and no data-path collective is involved."""
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
    local_ms = 10.0 + 5.0 * rank            # rank 1 is the slow replica
    ms = bench.max_over_ranks(local_ms, world, "cpu")
    out[rank] = (ms, bench.whole_job_gvoxels(world, 2 ** 28, ms))
    dist.barrier()
    dist.destroy_process_group()


def test_two_replicas_take_the_slowest_rank_and_sum_the_work():
    world, port = 2, 29731
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0][0] == res[1][0] == 15.0
    assert abs(res[0][1] - 2 * 2 ** 28 / 15e-3 / 1e9) < 1e-9


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(7.5, 1, "cpu") == 7.5
    assert abs(bench.whole_job_gvoxels(1, 10 ** 9, 1000.0) - 1.0) < 1e-12
