"""N>1 host logic of bench.py on CPU: world_size-2 gloo run of the max-over-ranks aggregation (weak scaling, replicas)."""
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
    ms, val = bench.aggregate_over_ranks(2.0 + 3.0 * rank, 1000, world)   # rank 1 is the slow one: 5 ms
    out[rank] = (ms, val)
    dist.barrier()
    dist.destroy_process_group()


def test_aggregate_is_max_over_ranks_and_whole_job_throughput():
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, 29517, out), nprocs=2, join=True)
    for r in (0, 1):
        ms, val = out[r]
        assert ms == 5.0 and abs(val - 2 * 1000 / 5e-3) < 1e-6


def test_aggregate_single_rank():
    sys.path.insert(0, ROOT)
    import bench
    ms, val = bench.aggregate_over_ranks(4.0, 1_000_000, 1)
    assert ms == 4.0 and val == 2.5e8
    assert abs(bench.alg_flops_per_element(0.7) - (8 * (6850 + 1600 * 0.7) + 600)) < 1e-9
