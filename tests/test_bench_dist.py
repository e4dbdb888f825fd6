"""N>1 host logic of bench.py on CPU (gloo, world_size 2): the max-over-ranks aggregation and the sharded arm's plumbing -
partition, exchange plan, the one all-gather of u on CPU tensors, unit accounting."""
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
    ms, val = bench.aggregate_over_ranks(2.0 + 3.0 * rank, 2000, world)   # rank 1 is the slow one: 5 ms; 2000 units in the job
    # the sharded arm of bench.py on CPU tensors: partition -> exchange plan -> all-gather of the owned slabs
    import numpy as np
    import synth
    from paper_2606_17390_b200 import shard
    cfg = synth.make_config(4, n=8)
    nn = cfg["coords"].shape[0]
    part = shard.partition(nn, cfg["conn"], world, rank)
    plan = shard.exchange_plan(part, torch.device("cpu"))
    u_owned = torch.from_numpy(cfg["u"][part["n0"]:part["n1"]].ravel().copy())
    ok = True
    for _ in range(3):                                           # the step's collective, repeated like the timed loop does
        ul = shard.exchange_u(u_owned, part, plan=plan)
        ok = ok and np.array_equal(ul.numpy().reshape(-1, 3), cfg["u"][part["lnodes"]])
    first = np.asarray(cfg["conn"])[part["elems"], 0]
    owned_elems = int(((first >= part["n0"]) & (first < part["n1"])).sum())      # every element is owned by exactly one rank
    out[rank] = (ms, val, ok, owned_elems, int(part["elems"].size), cfg["conn"].shape[0])
    dist.barrier()
    dist.destroy_process_group()


def test_aggregate_is_max_over_ranks_and_whole_job_throughput():
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, 29517, out), nprocs=2, join=True)
    for r in (0, 1):
        ms, val, ok, owned, local, ne = out[r]
        assert ms == 5.0 and abs(val - 2000 / 5e-3) < 1e-6
        assert ok and local < ne
    assert out[0][3] + out[1][3] == out[0][5]          # units of the whole job = elements of the one problem
    assert out[0][4] + out[1][4] > out[0][5]           # ghost layer recomputed on both sides


def test_aggregate_single_rank():
    sys.path.insert(0, ROOT)
    import bench
    ms, val = bench.aggregate_over_ranks(4.0, 1_000_000, 1)
    assert ms == 4.0 and val == 2.5e8
    assert abs(bench.alg_flops_per_element(0.7) - (8 * (6850 + 1600 * 0.7) + 600)) < 1e-9


def test_barlat_flop_model_is_the_frozen_one():
    """DESIGN.md section 10 / profiles/r02_ncu_full.md: elastic point 12,050 flop, plastic point 13,000 + 4,800 per Newton
    iteration; with the histogram measured at config 3 (Table 2 coefficients) that is 225.5 kflop per element."""
    sys.path.insert(0, ROOT)
    import bench
    hist = [0, 1, 3160, 91383, 2699726, 2703180, 171352, 3646, 571, 54]
    pf = sum(hist) / 8.0e6
    assert abs(bench.alg_flops_per_element_barlat(pf, hist) - 225.5e3) < 0.2e3
    assert bench.alg_flops_per_element_barlat(0.0, []) == 8 * 12050.0 + 600.0
    one_it = bench.alg_flops_per_element_barlat(1.0, [0, 0, 0, 8]) - bench.alg_flops_per_element_barlat(1.0, [0, 0, 8])
    assert abs(one_it - 8 * 4800.0) < 1e-6
